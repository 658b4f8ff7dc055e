"""CPU oracle for the MALA/SNAP grid bispectrum -- TEST INFRASTRUCTURE ONLY.

Thin ctypes wrapper around oracle/snap_oracle.c (see that file's header for the
passages of PAPER.md / SURVEY.md 8(c) it follows and for its pins).  Only
tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package; the product path never does.
"""
import ctypes as C
import os

import numpy as np

from .build import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build())
        _lib.oracle_cg.restype = C.c_double
        _lib.oracle_cg.argtypes = [C.c_int] * 6
        _lib.oracle_ntriples.restype = C.c_int
        _lib.oracle_usize.restype = C.c_int
        _lib.oracle_num_threads.restype = C.c_int
    return _lib


def _d(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t)) if a is not None else None


def ntriples(twojmax):
    return lib().oracle_ntriples(int(twojmax))


def triples(twojmax):
    """[n,3] doubled (j1,j2,j) in output order (Eq. (26))."""
    n = ntriples(twojmax)
    out = np.zeros((n, 3), dtype=np.int32)
    lib().oracle_triples(int(twojmax), _p(out, C.c_int))
    return out


def cg(J1, M1, J2, M2, J, M):
    """Clebsch-Gordan coefficient, all arguments doubled integers."""
    return lib().oracle_cg(int(J1), int(M1), int(J2), int(M2), int(J), int(M))


def wigner_D(J, a, b):
    """(J+1)x(J+1) complex D^J for the SU(2) element [[a,-conj b],[b,conj a]]."""
    ab = _d([a.real, a.imag, b.real, b.imag])
    out = np.zeros((J + 1, J + 1, 2), dtype=np.float64)
    lib().oracle_wigner_D(int(J), _p(ab, C.c_double), _p(out, C.c_double))
    return out[..., 0] + 1j * out[..., 1]


def pair(d, rcut, rfac0=0.99363, rmin0=0.0):
    """Returns (is_neighbor, a, b, fc) for displacement d = R_atom - r_point."""
    dd = _d(d)
    ab = np.zeros(4)
    fc = C.c_double(0.0)
    ok = lib().oracle_pair(_p(dd, C.c_double), C.c_double(rcut), C.c_double(rfac0), C.c_double(rmin0),
                           _p(ab, C.c_double), C.byref(fc))
    return bool(ok), complex(ab[0], ab[1]), complex(ab[2], ab[3]), fc.value


def usize(twojmax):
    return lib().oracle_usize(int(twojmax))


def uoff(J):
    return sum((K + 1) ** 2 for K in range(J))


def _sys_args(twojmax, rcutfac, rfac0, rmin0, wself, radelem, wj, pos, types, box, origin, pbc):
    radelem = _d(radelem).ravel()
    wj = _d(wj).ravel()
    assert radelem.shape == wj.shape
    pos = _d(pos).reshape(-1, 3)
    types = _i(types).ravel()
    assert types.shape[0] == pos.shape[0]
    box = _d(box).reshape(3, 3)
    origin = _d(origin).ravel()
    pbc = _i(pbc).ravel()
    keep = (radelem, wj, pos, types, box, origin, pbc)
    args = [C.c_int(int(twojmax)), C.c_double(rcutfac), C.c_double(rfac0), C.c_double(rmin0), C.c_double(wself),
            C.c_int(radelem.shape[0]), _p(radelem, C.c_double), _p(wj, C.c_double),
            C.c_int(pos.shape[0]), _p(pos, C.c_double), _p(types, C.c_int),
            _p(box, C.c_double), _p(origin, C.c_double), _p(pbc, C.c_int)]
    return args, keep


def bispectrum_points(points, pos, types, box, origin=(0, 0, 0), pbc=(1, 1, 1), *, twojmax=10, rcutfac=4.67637,
                      rfac0=0.99363, rmin0=0.0, wself=1.0, radelem=(0.5,), wj=(1.0,), triple_list=None,
                      want_imag=False, want_U=False, want_nbr=False, nbr_cap=256):
    """B at explicit Cartesian points.  Returns dict with 'B' [np,nt] and the optional extras:
    'imag' [np,nt], 'U' [np,usize] complex (levels packed, row-major [m'][m]),
    'nnbr' [np], 'nbr' [np,nbr_cap,5] = (c, q0, q1, q2, q3) per neighbor."""
    points = _d(points).reshape(-1, 3)
    npnt = points.shape[0]
    tr = triples(twojmax) if triple_list is None else _i(triple_list).reshape(-1, 3)
    nt = tr.shape[0]
    args, keep = _sys_args(twojmax, rcutfac, rfac0, rmin0, wself, radelem, wj, pos, types, box, origin, pbc)
    B = np.zeros((npnt, nt))
    imag = np.zeros((npnt, nt)) if want_imag else None
    usz = usize(twojmax)
    U = np.zeros((npnt, usz, 2)) if want_U else None
    nn = np.zeros(npnt, dtype=np.int32) if (want_nbr or True) else None
    nbr = np.zeros((npnt, nbr_cap, 5)) if want_nbr else None
    rc = lib().oracle_bispectrum_points(*args, C.c_int(npnt), _p(points, C.c_double), C.c_int(nt), _p(tr, C.c_int),
                                        _p(B, C.c_double), _p(imag, C.c_double), _p(U, C.c_double),
                                        _p(nn, C.c_int), _p(nbr, C.c_double), C.c_int(nbr_cap))
    if rc != 0:
        raise ValueError("oracle_bispectrum_points: invalid argument")
    res = {"B": B, "nnbr": nn, "triples": tr}
    if want_imag:
        res["imag"] = imag
    if want_U:
        res["U"] = U[..., 0] + 1j * U[..., 1]
    if want_nbr:
        res["nbr"] = nbr
    return res


def bispectrum_grid(pos, types, box, origin, pbc, ngrid, z_begin=0, z_end=None, *, twojmax=10, rcutfac=4.67637,
                    rfac0=0.99363, rmin0=0.0, wself=1.0, radelem=(0.5,), wj=(1.0,), sample=None):
    """out[(z_end-z_begin)*ny*nx, ncomp] (ix fastest), or out[len(sample), ncomp] for flat slab-relative
    point indices in `sample`."""
    ngrid = _i(ngrid).ravel()
    if z_end is None:
        z_end = int(ngrid[2])
    nt = ntriples(twojmax)
    args, keep = _sys_args(twojmax, rcutfac, rfac0, rmin0, wself, radelem, wj, pos, types, box, origin, pbc)
    if sample is not None:
        sample = np.ascontiguousarray(sample, dtype=np.int64).ravel()
        npnt = sample.shape[0]
        ns = C.c_long(npnt)
        sp = sample.ctypes.data_as(C.POINTER(C.c_long))
    else:
        npnt = (z_end - z_begin) * int(ngrid[1]) * int(ngrid[0])
        ns = C.c_long(0)
        sp = None
    out = np.zeros((npnt, nt))
    rc = lib().oracle_bispectrum_grid(*args, _p(ngrid, C.c_int), C.c_int(z_begin), C.c_int(z_end), ns, sp,
                                      _p(out, C.c_double))
    if rc != 0:
        raise ValueError("oracle_bispectrum_grid: invalid argument")
    return out


def gaussian_points(points, pos, types, box, origin=(0, 0, 0), pbc=(1, 1, 1), *, sigma, rcutfac=4.67637, radelem=(0.5,),
                    wj=(1.0,)):
    """Gaussian descriptors [np, ntypes] at explicit Cartesian points (snap_oracle.c for the reading)."""
    points = _d(points).reshape(-1, 3)
    radelem = _d(radelem).ravel()
    wj = _d(wj).ravel()
    pos = _d(pos).reshape(-1, 3)
    types = _i(types).ravel()
    box = _d(box).reshape(3, 3)
    origin = _d(origin).ravel()
    pbc = _i(pbc).ravel()
    out = np.zeros((points.shape[0], radelem.shape[0]))
    rc = lib().oracle_gaussian_points(C.c_double(rcutfac), C.c_double(sigma), C.c_int(radelem.shape[0]), _p(radelem, C.c_double),
                                      _p(wj, C.c_double), C.c_int(pos.shape[0]), _p(pos, C.c_double), _p(types, C.c_int),
                                      _p(box, C.c_double), _p(origin, C.c_double), _p(pbc, C.c_int),
                                      C.c_int(points.shape[0]), _p(points, C.c_double), _p(out, C.c_double))
    if rc != 0:
        raise ValueError("oracle_gaussian_points: invalid argument")
    return out


def grid_points(box, origin, ngrid, z_begin=0, z_end=None, sample=None):
    """Cartesian positions of the grid points of a slab in output order (ix fastest), or of flat indices `sample`."""
    box = _d(box).reshape(3, 3)
    nx, ny, nz = (int(v) for v in ngrid)
    if sample is None:
        z_end = nz if z_end is None else z_end
        idx = np.arange(z_begin * ny * nx, z_end * ny * nx)
    else:
        idx = np.asarray(sample, dtype=np.int64)
    ix, iy, iz = idx % nx, (idx // nx) % ny, idx // (nx * ny)
    return (_d(origin)[None, :] + (ix / nx)[:, None] * box[0] + (iy / ny)[:, None] * box[1] + (iz / nz)[:, None] * box[2])


def bj0j_grid(pos, types, box, origin, pbc, ngrid, z_begin=0, z_end=None, *, sample=None, twojmax=10, rcutfac=4.67637,
              rfac0=0.99363, rmin0=0.0, wself=1.0, radelem=(0.5,), wj=(1.0,)):
    """The 11 components B_{j,0,j} on a grid slab by the Chebyshev closed form (no Wigner-D, no CG): [npoints, twojmax+1];
    with `sample` (flat point indices relative to the slab) only those points: [len(sample), twojmax+1]."""
    nx, ny, nz = (int(v) for v in ngrid)
    z_end = nz if z_end is None else int(z_end)
    args, keep = _sys_args(twojmax, rcutfac, rfac0, rmin0, wself, radelem, wj, pos, types, box, origin, pbc)
    ng = _i([nx, ny, nz])
    smp = None if sample is None else np.ascontiguousarray(sample, dtype=np.int64)
    npts = (z_end - z_begin) * ny * nx if smp is None else smp.size
    out = np.zeros((npts, twojmax + 1))
    rc = lib().oracle_bj0j_grid(*args, _p(ng, C.c_int), C.c_int(int(z_begin)), C.c_int(z_end),
                                C.c_long(0 if smp is None else smp.size), _p(smp, C.c_long), _p(out, C.c_double))
    if rc != 0:
        raise ValueError("oracle_bj0j_grid: invalid argument")
    return out


def bispectrum_grad_points(points, pos, types, box, origin=(0, 0, 0), pbc=(1, 1, 1), *, beta=None, want_dB=True, twojmax=10,
                           rcutfac=4.67637, rfac0=0.99363, rmin0=0.0, wself=1.0, radelem=(0.5,), wj=(1.0,)):
    """Row f3 (Eq. (45)): dB[p, alpha, k, t] = d B_t(r_p) / d R_alpha,k by forward differentiation of the
    definition, and, with beta [npoints, ncomp], g[alpha, k] = sum_p sum_t beta[p, t] dB[p, alpha, k, t]."""
    points = _d(points).reshape(-1, 3)
    npnt = points.shape[0]
    nt = ntriples(twojmax)
    args, keep = _sys_args(twojmax, rcutfac, rfac0, rmin0, wself, radelem, wj, pos, types, box, origin, pbc)
    natoms = keep[2].shape[0]
    dB = np.zeros((npnt, natoms, 3, nt)) if want_dB else None
    b = None if beta is None else _d(beta).reshape(npnt, nt)
    g = np.zeros((natoms, 3)) if beta is not None else None
    rc = lib().oracle_bispectrum_grad_points(*args, C.c_int(npnt), _p(points, C.c_double), _p(dB, C.c_double), _p(b, C.c_double),
                                             _p(g, C.c_double))
    if rc != 0:
        raise ValueError("oracle_bispectrum_grad_points: invalid argument")
    return {"dB": dB, "g": g}


def num_threads():
    return lib().oracle_num_threads()


def set_num_threads(n):
    lib().oracle_set_num_threads(C.c_int(int(n)))
