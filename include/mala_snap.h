/*
 * mala_snap.h -- C ABI of libmala_snap.so: SNAP bispectrum descriptors on a real-space grid,
 * the data-parallel hot path of MALA inference (arXiv 2411.19617), hand-written CUDA for sm_100a.
 *
 * What is computed (PAPER.md = the paper text; SURVEY.md section 8 restates the mathematics):
 *   - neighbor density around each grid point, with cutoff, element weight and self term:
 *       Eq. (24)
 *   - its expansion coefficients u_j in 4-D hyperspherical harmonics:  Eq. (25)
 *   - the bispectrum B(r, j) = "scalar triple products of the expansion coefficients", real and
 *     rotation invariant:  PAPER.md:261;  number of components, Eq. (26)
 *   - evaluated at every point of the grid:
 *   - hyperparameters twojmax / rcutfac as in PAPER.md:597-599; f_c, theta0 map, rfac0, rmin0, wself as
 *     fixed by BASELINE.json north_star (DESIGN.md "Readings" #1-#6).
 *
 * Conventions
 *   - every pointer argument says HOST or DEVICE.  Host inputs are copied before the call returns.
 *   - angular momenta are DOUBLED integers (J = 2 j_true).
 *   - the library never aborts, throws or prints; non-zero return codes are
 *       MALA_SNAP_EINVAL  (-1)  invalid argument        (nothing was enqueued)
 *       MALA_SNAP_ECUDA   (-2)  CUDA runtime error      (message names the call)
 *       MALA_SNAP_ENOMEM  (-3)  host or device allocation failed
 *     and mala_last_error() returns a thread-local description of the last failure.
 *   - one handle must not be used by two host threads at once.  Calls on one handle are serialised on the device
 *     whatever streams they are given (the handle owns one workspace): a call waits, on the device, for the previous
 *     call on the same handle.  mala_snap_create / mala_snap_set_option("zi_impl") synchronise the device.
 *     There is no CPU fallback: without a CUDA device mala_snap_create fails with MALA_SNAP_ECUDA.
 */
#ifndef MALA_SNAP_H
#define MALA_SNAP_H

#ifdef __cplusplus
extern "C" {
#endif

#define MALA_SNAP_OK 0
#define MALA_SNAP_EINVAL (-1)
#define MALA_SNAP_ECUDA (-2)
#define MALA_SNAP_ENOMEM (-3)

/* largest supported twojmax.  Up to 10 a 32-point tile of U_tot fits one SM's shared memory; 11..14 run on half tiles. */
#define MALA_SNAP_MAX_TWOJMAX 14

typedef struct mala_snap mala_snap_t; /* opaque; owns device tables and a lazily grown workspace */

/*
 * Create a descriptor calculator (descriptor_type "Bispectrum", twojmax, rcutfac).
 *   handle   [out] HOST
 *   twojmax  0..MALA_SNAP_MAX_TWOJMAX (14), even or odd (10 in the paper's configurations; a hyperparameter)
 *   rcutfac  > 0; cutoff of type t is rcut_t = 2 * rcutfac * radelem[t]  (reading #10)
 *   rfac0    in (0, 1]: theta0 = rfac0 * pi * (r - rmin0) / (rcut_t - rmin0)      (north_star: 0.99363)
 *   rmin0    in [0, min rcut_t)                                                     (north_star: 0)
 *   wself    weight of the self term delta(0) of Eq. (24)                           (north_star: 1)
 *   ntypes   >= 1
 *   radelem  HOST [ntypes], > 0     (0.5 makes rcut = rcutfac, the MALA usage)
 *   wj       HOST [ntypes] element weights w_eta of Eq. (24)
 * Builds the triple list, Clebsch-Gordan tables and index lists on the host, uploads them, and computes
 * the constant zero-neighbor descriptor once.  Uses the current CUDA device.
 */
int mala_snap_create(mala_snap_t **handle, int twojmax, double rcutfac, double rfac0, double rmin0, double wself,
                     int ntypes, const double *radelem, const double *wj);

/* number of bispectrum components, Eq. (26) PAPER.md:263 (91 at twojmax = 10); < 0 on a NULL handle */
int mala_snap_ncomp(const mala_snap_t *h);

/* the (j1, j2, j) of every component, doubled, in output order (reading #7):
 *   for j1 = 0..twojmax, j2 = 0..j1, j = j1-j2 .. min(twojmax, j1+j2) step 2, if j >= j1.
 *   j1j2j  HOST [ncomp * 3] */
int mala_snap_triples(const mala_snap_t *h, int *j1j2j);

/*
 * Bispectrum descriptors on the z-slab [z_begin, z_end) of an nx x ny x nz grid.
 *   natoms   >= 0 (0 is valid: every point gets the self-term-only vector)
 *   pos      HOST [natoms*3] Cartesian, need not be wrapped into the cell (reading #14)
 *   types    HOST [natoms], 0-based, < ntypes
 *   box      HOST [9]  rows a1, a2, a3 of a general triclinic cell (either handedness)
 *   origin   HOST [3]  position of grid point (0,0,0); point (ix,iy,iz) sits at
 *                      origin + ix/nx a1 + iy/ny a2 + iz/nz a3                        (reading #8)
 *   pbc      HOST [3]  1 = periodic along a_i; all lattice images within the cutoff count, also an
 *                      atom's own images when the cell is smaller than the cutoff    (reading #13)
 *   ngrid    HOST [3]  nx, ny, nz > 0
 *   z_begin, z_end     0 <= z_begin <= z_end <= nz
 *   out      DEVICE [(z_end-z_begin)*ny*nx][ncomp] fp64, ix fastest, then iy, then iz; component k is
 *            triple k of mala_snap_triples.  No B0 subtraction, no normalisation (reading #6).
 *   cuda_stream  a cudaStream_t (NULL = default stream).  All device work is enqueued on it and the call
 *            returns without synchronising; `out` must stay alive until the stream has drained.
 * The slab is processed in internal chunks bounded by the workspace cap (see mala_snap_set_option).
 */
int mala_bispectrum_grid(mala_snap_t *h, int natoms, const double *pos, const int *types, const double box[9],
                         const double origin[3], const int pbc[3], const int ngrid[3], int z_begin, int z_end,
                         double *out, void *cuda_stream);

/*
 * Same, end to end with a HOST result: `out_host` is HOST memory [(z_end-z_begin)*ny*nx][ncomp]
 * (pinned memory makes the copies asynchronous with respect to the kernels).  The slab is computed in
 * z-chunks into two device staging buffers owned by the handle; the device->host copy of one chunk
 * overlaps the kernels of the next.  The call returns after the last copy has completed.
 */
int mala_bispectrum_grid_host(mala_snap_t *h, int natoms, const double *pos, const int *types,
                              const double box[9], const double origin[3], const int pbc[3], const int ngrid[3],
                              int z_begin, int z_end, double *out_host, void *cuda_stream);

/*
 * ---- the network that maps descriptors to the LDOS, fused behind the descriptor kernels ----------
 *
 * A fully connected feed-forward network, x_{l+1} = sigma(W_l x_l + b_l) (Eq. (19); neuron Eq. (18),
 * PAPER.md:164), applied point by point to the bispectrum vector to give the LDOS vector d(r, epsilon) (e.g.
 * 241 energy levels).  Runs on the tensor cores (tcgen05, TF32 operands rounded to nearest, fp32
 * accumulation, fp32 bias and activation); DESIGN.md section 13 states the tolerance against the fp64 oracle.
 *   nlayers        number of weight matrices, 1..8
 *   sizes          HOST [nlayers+1]: widths w_0 .. w_L, each 1..256 (w_0 = number of descriptor components for the fused call)
 *   weights        HOST [nlayers] pointers; weights[l] is W_l, [sizes[l+1]][sizes[l]] row-major fp64 (row = output neuron)
 *   biases         HOST [nlayers] pointers; biases[l] is b_l, [sizes[l+1]] fp64
 *   activation     sigma: 0 identity, 1 ReLU, 2 leaky ReLU (slope 0.01), 3 logistic sigmoid              (reading N2)
 *   activate_last  1: sigma follows the last layer too, as Eq. (19) is written; 0: linear output layer     (reading N1)
 *   in_shift, in_scale  HOST [sizes[0]] or NULL: the input scaling x_0 = (x - shift) * scale of PAPER.md:473 (reading N3)
 * All host arrays are copied (and the weights rounded to TF32 and packed) before the call returns.
 */
typedef struct mala_mlp mala_mlp_t;
int mala_mlp_create(mala_mlp_t **net, int nlayers, const int *sizes, const double *const *weights, const double *const *biases,
                    int activation, int activate_last, const double *in_shift, const double *in_scale);

/* input / output width of the network (either pointer may be NULL) */
int mala_mlp_widths(const mala_mlp_t *net, int *w_in, int *w_out);

/*
 * The network alone:  y[p][w_L] = net(x[p][w_0])  for npoints rows.
 *   x   DEVICE [npoints][w_0] fp64          y   DEVICE [npoints][w_L] fp32
 * Enqueued on cuda_stream; does not synchronise.
 */
int mala_mlp_forward(mala_mlp_t *net, long long npoints, const double *x, float *y, void *cuda_stream);

/* NULL-safe */
void mala_mlp_destroy(mala_mlp_t *net);

/*
 * Descriptors and network in one call: the LDOS on the z-slab [z_begin, z_end) of the grid.  All arguments but `net` and
 * `ldos` as mala_bispectrum_grid.  Per workspace chunk the descriptors go to a compact device staging buffer owned by the
 * handle and the network consumes them before the next chunk starts; they are never written to caller memory.
 *   ldos  DEVICE [(z_end-z_begin)*ny*nx][w_L] fp32, ix fastest
 * MALA_SNAP_EINVAL if the network's input width is not mala_snap_ncomp(h).  Enqueued on cuda_stream; does not synchronise.
 * mala_snap_kernel_times reports the network under ms[3].
 */
int mala_bispectrum_ldos_grid(mala_snap_t *h, mala_mlp_t *net, int natoms, const double *pos, const int *types,
                              const double box[9], const double origin[3], const int pbc[3], const int ngrid[3], int z_begin,
                              int z_end, float *ldos, void *cuda_stream);

/*
 * ---- the adjoint of the descriptor map (forces) --------------------------------------------------
 *
 * "Apply dB(r, j; R)/dR_alpha to an array" -- the third factor of the chain rule for the force on ion alpha, Eqs. (44)-(45),
 * PAPER.md:418-428.  With beta(r, j) = dE/dB(r, j) supplied by the caller (the result of back-propagating through the
 * network),
 *     g[alpha][k] += sum_{grid points r of the slab} sum_j beta[r][j] * dB(r, j)/dR_{alpha,k},     k = x, y, z,
 * where all periodic images of atom alpha move with it.  The force contribution is f_alpha = -g[alpha].
 *   beta   DEVICE [(z_end-z_begin)*ny*nx][ncomp] fp64, ix fastest (the layout of mala_bispectrum_grid's out)
 *   g      DEVICE [natoms*3] fp64; the call ADDS the slab's contribution (zero it before the first slab; slabs and GPUs sum)
 * All other arguments as mala_bispectrum_grid.  twojmax <= 10 (MALA_SNAP_EINVAL above).  Enqueued on cuda_stream; does not
 * synchronise.  The per-atom sums use floating-point atomics: results are reproducible to rounding, not bit for bit (Y itself is
 * accumulated in fixed point and does not depend on the order of the additions; see "yi_impl").
 * mala_snap_kernel_times reports compute_yi under ms[2] and compute_dedr under ms[3].
 */
int mala_bispectrum_force_adjoint(mala_snap_t *h, int natoms, const double *pos, const int *types, const double box[9],
                                  const double origin[3], const int pbc[3], const int ngrid[3], int z_begin, int z_end,
                                  const double *beta, double *g, void *cuda_stream);

/*
 * Gaussian descriptors on the same grid ("a sum of Gaussians centered at R", the Gaussian representation of
 * the ionic configuration behind Eqs. (40)-(43)).  One channel per atom type t:
 *     G_t(r) = wj[t] * (2 pi sigma^2)^(-3/2) * sum exp(-|R - r|^2 / (2 sigma^2))
 * over the atoms of type t and their periodic images with |R - r| < rcut_t (the handle's cutoffs; strict).  The paper
 * fixes neither the normalisation nor the truncation: this is DESIGN.md reading G1.  twojmax of the handle is not used.
 *   sigma    > 0, the Gaussian width w_G of PAPER.md:416, in the length unit of pos
 *   out      DEVICE [(z_end-z_begin)*ny*nx][ntypes] fp64, ix fastest; all other arguments as mala_bispectrum_grid
 * At most 4 atom types (MALA_SNAP_EINVAL otherwise).  Work is enqueued on cuda_stream; the call does not synchronise.
 */
int mala_gaussian_grid(mala_snap_t *h, double sigma, int natoms, const double *pos, const int *types, const double box[9],
                       const double origin[3], const int pbc[3], const int ngrid[3], int z_begin, int z_end, double *out,
                       void *cuda_stream);

/*
 * mala_gaussian_grid for callers that must not allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): same arguments, same result up to rounding, but the call makes no cudaMalloc /
 * cudaMallocAsync / cudaFree and uses no allocating library routine.  Its scratch (ghost atoms, cell list, counters and the
 * neighbor-candidate lists of tile_bin_kernel) is a file-scope static device array of MALA_SNAP_STATIC_SCRATCH_BYTES (16 MiB)
 * that every GPU loading the library holds until exit; the handle resolves its device address once, in mala_snap_create.
 *   limit    the ghost atoms of the slab (32 bytes each), the cell list (4 bytes per cell) and the candidate lists of one
 *            tile per SM must fit the array; the grid is then walked in as many chunks as it takes.  Beyond that the call
 *            returns MALA_SNAP_EINVAL with the byte counts in mala_last_error() and enqueues nothing: use
 *            mala_gaussian_grid, or smaller z-slabs.  Config 2 (256 atoms, 90^3 points) needs about 3 % of the array.
 *   sharing  ONE array per GPU (and process), shared by every handle and every call of this entry point, and it keeps the
 *            last call's contents (the call clears the counters that must start at zero).  Calls on one handle are
 *            serialised as everywhere else, but calls on DIFFERENT handles of one process that overlap on the GPU race on
 *            the array: order them (one stream, or events).
 * The device of the handle must be current (MALA_SNAP_EINVAL otherwise).  Host memory (the ghost list) is still taken from
 * the C++ heap; positions are read from pageable host memory as in every other entry point.
 */
#define MALA_SNAP_STATIC_SCRATCH_BYTES (16u << 20)
int mala_gaussian_grid_static(mala_snap_t *h, double sigma, int natoms, const double *pos, const int *types, const double box[9],
                              const double origin[3], const int pbc[3], const int ngrid[3], int z_begin, int z_end, double *out,
                              void *cuda_stream);

/*
 * Tuning / test knobs.  Unknown names give MALA_SNAP_EINVAL.
 *   "zi_impl"          0 = automatic (register-tiled block kernel; on 16-point half tiles above twojmax 10),
 *                      1 = generic table-driven kernel (twojmax <= 10), 2 = per-triple specialised kernel (EINVAL if
 *                      twojmax != 10), 3 = anti-diagonal kernel (code specialised on j1 only, any twojmax), 4 = block kernel
 *                      (any twojmax).  All tables but the per-triple kernel's are per-handle arrays in global memory, so
 *                      handles of different twojmax coexist.  Every kernel gives the same B up to rounding (summation order).
 *   "ui_impl"          0 = automatic (twojmax 8..14: pipelined sampling kernel; twojmax 1..7: sampling kernel;
 *                      twojmax 0: column kernel), 1 = column kernel (polynomial recursion, accumulators in shared memory; any
 *                      twojmax), 2 = sampling kernel (column polynomials evaluated at the roots of unity, sums in registers,
 *                      inverse DFT per tile; EINVAL outside 1..10), 3 = pipelined sampling kernel (a producer warp prepares
 *                      the neighbor queue of the next tile; EINVAL below 8)
 *   "yi_impl"          compute_yi of mala_bispectrum_force_adjoint: 0 = automatic (2), 1 = table-driven kernel (element by
 *                      element), 2 = register-tiled block kernel with Y accumulated in 60-bit fixed point by native 32-bit
 *                      shared-memory atomics (a power-of-two scale per grid point; Y does not depend on the order of the warps;
 *                      rounding about 1e-12 of the largest |Y| of a grid point), 3 = the same kernel with fp64 atomics (compare-and-
 *                      swap loops on sm_100a; rounding 1e-14, order-dependent)
 *   "dedr_impl"        compute_dedr of mala_bispectrum_force_adjoint: 0 = sampling kernel (the DFT of Y's columns as the
 *                      coefficients of a polynomial in the pair's sample values; twojmax 1..10, default), 1 = column kernel
 *   "timing"           1 = record a CUDA-event pair on the caller's stream around every kernel launch of the
 *                      following calls (read back with mala_snap_kernel_times); 0 = off (default)
 *   "workspace_mb"     cap, in MiB, of the U_tot + candidate workspace (default 4096)
 *   "cand_cap_limit"   test hook: clamp the per-tile candidate capacity to this value (0 = off, default).  A value below
 *                      the true bound makes tile_bin_kernel overflow, which must surface as MALA_SNAP_ECUDA (see
 *                      mala_snap_last_stats); never set it in production
 *   "host_chunk_mb"    cap, in MiB, of each of the two staging buffers of mala_bispectrum_grid_host (default 256;
 *                      outputs above 96 MiB go in chunks that shrink -- a third of what is left, whole tile layers, at least
 *                      eight planes -- so that the copy of one chunk overlaps the kernels of the next and the last, exposed
 *                      copy is short)
 */
int mala_snap_set_option(mala_snap_t *h, const char *name, long long value);

/*
 * Counters of the last mala_bispectrum_grid* call on this handle (HOST array of 8):
 *   [0] kernels launched   [1] chunks   [2] tiles   [3] ghost atoms (atoms + periodic images kept)
 *   [4] candidate capacity per tile   [5] workspace bytes in use   [6] points
 *   [7] status bits of the handle (0 = healthy; bit 0: a neighbor-candidate list overflowed its host-computed bound and was
 *       truncated, i.e. results of that call are invalid)
 * Waits for the last call on the handle (its status word is part of the answer) and returns MALA_SNAP_ECUDA when a status
 * bit is set.  A raised bit is sticky: every later mala_*_grid call on the handle fails with MALA_SNAP_ECUDA at entry as soon
 * as the offending call has drained; mala_bispectrum_grid_host, which synchronises anyway, reports it on return.
 */
int mala_snap_last_stats(mala_snap_t *h, long long stats[8]);

/*
 * Measurement: device time of the kernels of the last mala_bispectrum_grid* call on this handle, by class, from
 * the event pairs recorded when the "timing" option is on (rows of SURVEY.md 8(a)):
 *   ms[0] tile_bin (a2 + constant fill of empty tiles)   ms[1] compute_ui (a3 + a4)
 *   ms[2] compute_zi_bi (a5 + a6 + a7)                    ms[3] other (test hooks)
 *   launches[k] = number of launches summed into ms[k].   Both HOST arrays of 4.
 * Waits for those events (so for the call's work).  All zeros if timing was off.
 */
int mala_snap_kernel_times(mala_snap_t *h, double ms[4], long long launches[4]);

/* Measurement: name of the compute_zi / compute_bi kernel the handle launches with its current options (the kernel the
 * roofline of bench.py is reported for); a static string, "" on a NULL handle */
const char *mala_snap_zi_kernel(const mala_snap_t *h);

/*
 * Measurement: achieved FP64 FMA rate of this device (TFLOP/s, 2 flop per DFMA) from a register-only
 * microbenchmark -- 8 independent FMA chains per thread, 4 CTAs of 256 threads per SM, best of 5 timed launches
 * after one warm-up -- the measured denominator of the FP64 roofline.
 *   tflops            [out] HOST
 *   sm_mhz_effective  [out] HOST, may be NULL: the SM clock that rate implies at 64 DFMA/clk/SM
 * Synchronises the stream.
 */
int mala_snap_fp64_peak(double *tflops, double *sm_mhz_effective, void *cuda_stream);

/*
 * Test hook: the Clebsch-Gordan coefficient the library's own table generator produces (doubled arguments).
 * Pure host arithmetic; lets the CPU-only test-suite check the tables without a GPU.
 */
double mala_snap_clebsch_gordan(int J1, int M1, int J2, int M2, int J, int M);

/*
 * Test hook: U_tot (Eq. (25) coefficients, summed over neighbors, self term included) at the grid points of
 * one z-slab, in the library's internal half-column storage:
 *   u_out  DEVICE [npoints][nelem][2] fp64 (re, im), nelem = sum_J (J+1)*(J/2+1); element (J, mb <= J/2, ma)
 *          at index sum_{K<J}(K+1)*(K/2+1) + mb*(J+1) + ma.
 * Returns nelem (>0) on success.  Synchronises the stream.
 */
int mala_snap_debug_utot(mala_snap_t *h, int natoms, const double *pos, const int *types, const double box[9],
                         const double origin[3], const int pbc[3], const int ngrid[3], int z_begin, int z_end,
                         double *u_out, void *cuda_stream);

/* NULL-safe; frees tables, workspace and staging buffers */
void mala_snap_destroy(mala_snap_t *h);

/* thread-local message for the last non-zero return on this thread ("" if none) */
const char *mala_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* MALA_SNAP_H */
