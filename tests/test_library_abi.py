"""CPU-only checks of the C-ABI library: it loads, exports every symbol include/mala_snap.h declares, and its host-side
table generator agrees with the oracle's independent one.  No compute call is made (there is no GPU here)."""
import ctypes
import os
import re

import numpy as np
import pytest

import oracle
import paper_2411_19617_b200 as pkg
from paper_2411_19617_b200 import snap as binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "mala_snap.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(mala_[a-z_0-9]+)\s*\(", text)))


def test_header_symbols_are_exported_and_bound():
    names = _declared_symbols()
    assert "mala_snap_create" in names and "mala_bispectrum_grid" in names and "mala_snap_destroy" in names
    lib = ctypes.CDLL(pkg.library_path()) if os.path.exists(pkg.library_path()) else pkg.load_library()
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/mala_snap.h but not exported"
    assert sorted(binding.EXPORTS) == names


def test_library_is_sm100a_and_has_tma():
    """cuobjdump shows an sm_100a cubin; UBLKCP is the SASS of the cp.async.bulk U_tot tile load."""
    import shutil
    import subprocess
    exe = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(exe):
        pytest.skip("cuobjdump not available")
    pkg.load_library()
    lst = subprocess.run([exe, "-lelf", pkg.library_path()], capture_output=True, text=True).stdout
    assert "sm_100a" in lst
    sass = subprocess.run([exe, "-sass", pkg.library_path()], capture_output=True, text=True).stdout
    assert "UBLKCP" in sass and "DFMA" in sass


def test_create_without_gpu_fails_loudly():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(pkg.MalaSnapError) as e:
        pkg.MalaSnap()
    assert e.value.code == binding.MALA_SNAP_ECUDA
    assert "no CPU fallback" in str(e.value)


def test_create_argument_errors_come_before_device_use():
    lib = pkg.load_library()
    h = ctypes.c_void_p()
    one = (ctypes.c_double * 1)(0.5)
    bad = [dict(twojmax=-1), dict(twojmax=15), dict(rcutfac=0.0), dict(rfac0=0.0), dict(rfac0=1.5), dict(rmin0=5.0), dict(ntypes=0)]
    for kw in bad:
        a = dict(twojmax=10, rcutfac=4.676, rfac0=0.99363, rmin0=0.0, wself=1.0, ntypes=1)
        a.update(kw)
        rc = lib.mala_snap_create(ctypes.byref(h), a["twojmax"], a["rcutfac"], a["rfac0"], a["rmin0"], a["wself"], a["ntypes"], one, one)
        assert rc == binding.MALA_SNAP_EINVAL, kw
        assert pkg.mala_last_error() != ""
    assert lib.mala_snap_ncomp(None) < 0
    lib.mala_snap_destroy(None)  # NULL-safe


@pytest.mark.parametrize("tj", [0, 1, 2, 3, 5, 10, 14])
def test_library_cg_table_matches_oracle_racah(tj):
    """two independent implementations (long-double factorial table vs the oracle's) of the same closed form"""
    worst = 0.0
    for J1 in range(tj + 1):
        for J2 in range(J1 + 1):
            for J in range(J1 - J2, min(tj, J1 + J2) + 1, 2):
                for M1 in range(-J1, J1 + 1, 2):
                    for M2 in range(-J2, J2 + 1, 2):
                        M = M1 + M2
                        if abs(M) > J:
                            continue
                        a = pkg.mala_snap_clebsch_gordan(J1, M1, J2, M2, J, M)
                        b = oracle.cg(J1, M1, J2, M2, J, M)
                        worst = max(worst, abs(a - b))
    assert worst < 5e-15


def test_workload_generators_are_seeded_and_shaped():
    from paper_2411_19617_b200 import workloads
    for cfg, natoms, npts in ((1, 4, 18 ** 3), (2, 256, 90 ** 3), (3, 256, 100 ** 3), (4, 40, 160 ** 3)):
        a, b = workloads.make(cfg), workloads.make(cfg)
        assert a.pos.shape == (natoms, 3) and a.npoints == npts
        assert np.array_equal(a.pos, b.pos)
    w3 = workloads.make(3)
    L = w3.box[0, 0]
    d = w3.pos[:, None, :] - w3.pos[None, :, :]
    d -= L * np.round(d / L)
    r = np.sqrt((d ** 2).sum(-1)) + 10 * np.eye(256)
    assert r.min() >= 2.3 and abs(256 / L ** 3 - 0.0530) < 1e-6
