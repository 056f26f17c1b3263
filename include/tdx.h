/* tdx.h -- C ABI of libtdx.so: B200 (sm_100a) batched tridiagonal line solves along the x, y and z lines of a
 * 3-D staggered grid by the Parallel Diagonal Dominant (PDD) and Parallel Partition (PPT) methods of
 * Ha, Park & You, arxiv 1812.01178 (Section 3.2; Algorithm 1), used INSIDE one GPU:
 * P partitions per line are solved by independent threads, coupled through the reduced interface system Z.
 *
 * Conventions (all entry points)
 *   - fp64 throughout (the paper's precision).
 *   - Field layout: x fastest, idx(i,j,k) = i + nx*(j + ny*k), 0-based, contiguous, base 16-byte aligned.
 *     A line along dir has length n_dir and stride 1 (x), nx (y), nx*ny (z).  No transpose is ever made
 *     (the point of the paper, L51-74).
 *   - Solves are IN PLACE: the right-hand side is overwritten by the solution.
 *   - Pointers marked HOST are read during the call and never retained; pointers marked DEVICE must be valid on
 *     the grid's device and belong to the caller (e.g. torch.Tensor.data_ptr()).  The library never frees them.
 *   - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  Device entry points are
 *     asynchronous with respect to the host; plan tables are built on first use on the same stream (that first call
 *     allocates and synchronises).  With its plan in the cache a sweep or Helmholtz solve is plain stream work -- no
 *     allocation, no synchronisation -- and may be recorded by CUDA stream capture (one warm-up call outside the capture).
 *   - Every call returns tdx_status_t.  Argument validation precedes any launch: on an argument error nothing
 *     is written.  tdx_last_error() gives a thread-local message for the last failure on this thread.
 *   - There is no CPU fallback and no other backend: without a CUDA device every solve returns TDX_ERR_CUDA.
 *   - A grid object caches its plans (at most 64; the oldest are dropped) and is NOT safe for concurrent calls from
 *     several host threads: use one grid per thread.  Different grids are independent.
 */
#ifndef TDX_H
#define TDX_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct tdx_grid tdx_grid_t;                 /* opaque; owns grid metrics and cached plan tables */

typedef enum { TDX_DIR_X = 0, TDX_DIR_Y = 1, TDX_DIR_Z = 2 } tdx_dir_t;
/* THOMAS: one thread per line, plain Thomas recurrence (GPU baseline; P ignored).
 * PDD   : PAPER.md L148-154 -- far-end spike entries of Z dropped, 2x2 interface blocks (Alg.1 step 5).
 * PPT   : PAPER.md L126-146, L156 -- Z solved exactly (to rounding).                                  */
typedef enum { TDX_MODE_THOMAS = 0, TDX_MODE_PDD = 1, TDX_MODE_PPT = 2 } tdx_mode_t;
typedef enum { TDX_BC_DIRICHLET = 0, TDX_BC_PERIODIC = 1, TDX_BC_NEUMANN = 2 } tdx_bc_t;
/* Where the unknowns of a direction sit on the staggered grid (velocities at faces, pressure at centres). */
typedef enum { TDX_LOC_CENTER = 0, TDX_LOC_FACE = 1 } tdx_loc_t;
typedef enum {
    TDX_OK = 0,
    TDX_ERR_INVALID_ARG = -1,      /* null pointer, bad enum, non-increasing faces, n < 2 ...            */
    TDX_ERR_BAD_PARTITION = -2,    /* P < 1, P > TDX_MAX_P or floor(n_dir/P) < 2                          */
    TDX_ERR_ALLOC = -3,
    TDX_ERR_CUDA = -4,             /* no device / launch or runtime failure (text in tdx_last_error)      */
    TDX_ERR_UNSUPPORTED = -5,      /* valid request this build cannot run (text in tdx_last_error)        */
    TDX_ERR_PDD_BOUND = -6         /* strict PDD checking is on (tdx_grid_set_pdd_strict) and the a-priori bound of this
                                      (dir, P, operator) exceeds the limit; nothing was launched           */
} tdx_status_t;

#define TDX_MAX_P 1024             /* partitions per line                                                 */
#define TDX_MAX_ROWS_PER_PARTITION 64   /* rows one THREAD keeps in registers.  Not a limit on the caller's P: longer
                                           partitions are cut again into sub-partitions inside the thread block (two-level
                                           PDD / PPT; at most 256 sub-partitions per line), with the
                                           result of the caller's P: PPT exact, PDD = PDD with his P partitions.     */

/* Create a grid.  xf/yf/zf: HOST arrays of n+1 strictly increasing face coordinates per direction (copied).
 * Metrics (reading A3): width D_j, centre spacings hm_j, hp_j, mirrored ghost at Dirichlet/Neumann
 * ends, wrap-around at periodic ends; delta2 u_j = [(u_{j+1}-u_j)/hp_j - (u_j-u_{j-1})/hm_j]/D_j.
 * device: CUDA ordinal.  On success *out owns device memory until tdx_grid_destroy.                      */
tdx_status_t tdx_grid_create(int nx, int ny, int nz,
                             const double* xf, const double* yf, const double* zf,
                             tdx_bc_t bcx, tdx_bc_t bcy, tdx_bc_t bcz,
                             int device, tdx_grid_t** out);
tdx_status_t tdx_grid_destroy(tdx_grid_t* grid);   /* frees plan tables; NULL is accepted                 */

/* Strict PDD checking ("when n >> p", L164, L172).  PDD never falls back silently: it runs as
 * asked.  With max_dropped > 0 every later PDD solve on this grid whose a-priori bound -- the largest far spike end
 * |v_last|, |w_first| that PDD deletes from Z, tdx_pdd_dropped_bound -- exceeds max_dropped returns TDX_ERR_PDD_BOUND
 * before anything is launched (1e-11 keeps the result within 1e-10 of the exact solution, reading A9).
 * Helmholtz solves with per-line shifts are judged by their least dominant line (smallest kx2 + kz2); slabs by the
 * rank-level bound.  0 switches the check off (the default).  THOMAS / PPT are never refused.               */
tdx_status_t tdx_grid_set_pdd_strict(tdx_grid_t* grid, double max_dropped);

/* Partition map (host, integer only; bit-exact contract, reading A5): q = n/P, r = n%P,
 * starts[p] = p*q + min(p,r), p = 0..P.  The paper has only m = n/p.
 * starts: HOST array of P+1 ints.                                                                        */
tdx_status_t tdx_partition_bounds(int n, int P, int* starts);

/* ADI sweep (Algorithm 1): solve (I - alpha*delta2_dir) x = rhs on every line of
 * direction dir, in place.  Rows satisfy |b| = |a| + |c| + 1 (L162).  Periodic directions: THOMAS closes the line by
 * Sherman-Morrison (Eq.(3) with a rank-1 update); PDD and PPT (P <= 128) put the two wrap-around corner entries into
 * Delta A (L78-91), i.e. P interfaces and a cyclic reduced system Z -- Woodbury, Eq.(3)-(4): exact for PPT, and PDD deletes
 * the far spike ends of every partition (reading A16: an approximation already at P = 2).
 * rhs_inout: DEVICE, nx*ny*nz doubles.  P: partitions per line (ignored for THOMAS), 1 <= P <= TDX_MAX_P,
 * floor(n_dir / P) >= 2, any partition length (see TDX_MAX_ROWS_PER_PARTITION).  In PDD the result depends on P (the
 * dropped couplings) and the caller's partition map is used as given; in PPT it does not, and the library
 * may run with coarser partitions than asked for: fewer than 8 rows per partition are merged pairwise up to 8, x lines whose
 * partition length the bulk-copy kernel cannot take are cut into 16-row ones (tdx_last_launch shows the shape used).  */
tdx_status_t tdx_adi_sweep(tdx_grid_t* grid, tdx_dir_t dir, tdx_mode_t mode, int P,
                           double alpha, double* rhs_inout, void* stream);

/* The same sweep with the unknowns of direction dir at cell centres (TDX_LOC_CENTER: identical to tdx_adi_sweep) or at
 * cell faces (TDX_LOC_FACE; SURVEY 8(f) N1 -- the wall-normal velocity component of the ADI step).
 * Face unknowns: row i of a line is the value at face f_{i+1}; delta2 v_i = [(v_{i+1}-v_i)/Da - (v_i-v_{i-1})/Db]/hc with
 * the adjacent cell widths Db, Da and hc = (Db+Da)/2.  Dirichlet: both walls carry 0, row n-1 is the wall face and is an
 * identity row (its right-hand side passes through); periodic: every row regular.  Neumann ends or n < 3:
 * TDX_ERR_UNSUPPORTED.  rhs_inout: DEVICE, nx*ny*nz doubles. */
tdx_status_t tdx_adi_sweep_at(tdx_grid_t* grid, tdx_dir_t dir, tdx_loc_t loc, tdx_mode_t mode, int P,
                              double alpha, double* rhs_inout, void* stream);

/* One ADI step for ncomp fields stored back to back ([ncomp][nz][ny][nx], e.g. the three velocity components that
 * Algorithm 1 batches): x sweep, then y sweep, then z sweep of (I - alpha*delta2) over all components,
 * one launch per direction for each run of consecutive components with the same location.  loc: HOST, ncomp*3 ints
 * loc[c*3 + dir] in {TDX_LOC_CENTER, TDX_LOC_FACE}, or NULL for all centres (staggered velocities: u = face in x,
 * v = face in y, w = face in z).  All plans are validated before the first launch.  rhs_inout: DEVICE. */
tdx_status_t tdx_adi_step(tdx_grid_t* grid, tdx_mode_t mode, int Px, int Py, int Pz, double alpha,
                          int ncomp, const int* loc, double* rhs_inout, void* stream);

/* Poisson y-solves after the spanwise transform: for every wavenumber m < nm and
 * x-index i solve (delta2_y - lambda) phi = rhs with lambda = kx2[i] + kz2[m] >= 0, Neumann ends;
 * |b| = |a| + |c| + lambda (L172).  Lines with lambda == 0 exactly are singular and are pinned at j = 0
 * (b_0 := 1, c_0 := 0, d_0 := 0).  kz2: HOST, nm doubles.  kx2: HOST, nx doubles, or NULL for zeros
 * A kx2 with non-zero entries gives every line its own matrix (the paper's cosine-x / Fourier-z solve): factorisation,
 * spikes and reduced system are then computed on the fly per line; THOMAS takes any shape (device workspace of nx*ny*nm
 * doubles owned by the grid); PPT takes any P (partitions of more than 16 rows are cut again inside the thread block --
 * the result is exact either way, L156); PDD takes at most 16 rows per partition, ceil(ny/P) <= 16 (else
 * TDX_ERR_UNSUPPORTED: raise P).  Asynchronous like the shared-matrix case: kx2 / kz2 are copied to the device (and cached
 * by content) before the call returns.
 * rhs_inout: DEVICE, complex128 interleaved [nm][ny][nx] (x fastest) = 2*nm*ny*nx doubles; the matrix is
 * real, so re and im are two right-hand sides of one factorisation.                                       */
tdx_status_t tdx_helmholtz_wavenumber_solve(tdx_grid_t* grid, tdx_mode_t mode, int P,
                                            int nm, const double* kx2, const double* kz2,
                                            double* rhs_inout, void* stream);

/* Transforms around the Poisson y-solves ("half-range cosine transform in the streamwise x-direction and
 * Fourier transform in the spanwise z-direction ... after which the pseudo-pressure is obtained via inverse
 * transforms").  All DEVICE buffers, 16-byte aligned, fp64, no transpose, asynchronous on `stream`.
 *
 * tdx_dct_x: in place on field [nz][ny][nx].  inverse == 0: X_k = sum_n x_n cos(pi k (n + 1/2) / nx), k < nx
 * (cell-centred values, Neumann walls; unnormalised).  inverse != 0: x_n = (1/nx)[X_0 + 2 sum_{k>=1} X_k cos(...)],
 * the exact inverse.  nx = 2^k in [16, 4096] or 3*2^k in [48, 3072], else TDX_ERR_UNSUPPORTED.
 *
 * tdx_rfft_z: field_in real [nz][ny][nx] -> spec_out complex128 interleaved [nz/2+1][ny][nx] (the layout
 * tdx_helmholtz_wavenumber_solve takes), F_m = sum_k f_k exp(-2 pi i m k / nz).  tdx_irfft_z: the inverse including
 * the 1/nz (imaginary parts of F_0 and F_{nz/2} do not enter).  Out of place (in == out is TDX_ERR_INVALID_ARG); the
 * input is not modified.  nz = 2^k in [16, 1024] or 3*2^k in [48, 1536], and nx even, else TDX_ERR_UNSUPPORTED.  */
tdx_status_t tdx_dct_x(tdx_grid_t* grid, int inverse, double* field_inout, void* stream);
tdx_status_t tdx_rfft_z(tdx_grid_t* grid, const double* field_in, double* spec_out, void* stream);
tdx_status_t tdx_irfft_z(tdx_grid_t* grid, const double* spec_in, double* field_out, void* stream);

/* Direct Poisson solve of PAPER.md:L45 / L170-174 in the paper's order: cosine transform in x, Fourier transform in z,
 * the y-solves (delta2_y - kx2[i] - kz2[m]) phi^ = f^ (Neumann ends, mode (0,0) pinned at j = 0), inverse Fourier,
 * inverse cosine: five passes over the field.  field_inout: DEVICE [nz][ny][nx], f in, phi out.  spec_work: DEVICE
 * scratch of 2*(nz/2+1)*ny*nx doubles (caller-owned).  kx2 (HOST, nx) / kz2 (HOST, nz/2+1): the modified wavenumbers,
 * or NULL for kx2[i] = 2(1-cos(pi i/nx))/dx^2, kz2[m] = 2(1-cos(2 pi m/nz))/dz^2 of the grid's uniform x / z spacing
 * (TDX_ERR_UNSUPPORTED if that direction is not uniform).  mode / P: as tdx_helmholtz_wavenumber_solve with per-line
 * shifts (PDD needs ceil(ny/P) <= 16; the paper uses PPT here because PDD is inaccurate on the weakly
 * dominant low modes, L172).  Every argument check of every stage precedes the first launch.  Asynchronous on
 * `stream` like every device entry point: all five stages are enqueued, nothing waits for them; kx2 / kz2 (or the
 * grid's own wavenumbers) are on the device, cached by content, when the call returns.                        */
tdx_status_t tdx_poisson_solve(tdx_grid_t* grid, tdx_mode_t mode, int P, const double* kx2, const double* kz2,
                               double* field_inout, double* spec_work, void* stream);

/* The paper's decomposition one level up (Algorithm 1 L222-258, L156/L174): the field is
 * cut into slabs along `dir` (y in the paper; z also taken), one slab per GPU / rank, and every rank is ONE partition
 * of the PDD or PPT method; inside the rank the slab's lines are solved by the intra-GPU sweeps above.
 *
 * tdx_slab_create: `slab_grid` describes this rank's slab (its extent along dir = the rank's share of n_global under
 * the partition map of tdx_partition_bounds(n_global, nranks); the other two extents are the whole domain's; the
 * grid's own faces / boundary condition along dir are not used).  faces_global: HOST, n_global+1 face coordinates of
 * the whole line; bc_global: Dirichlet or Neumann (a periodic slab direction is TDX_ERR_UNSUPPORTED); alpha as in
 * tdx_adi_sweep; across: PDD (neighbour exchange, exact where the spikes have decayed, L148-154) or PPT (all-gather,
 * exact, L126-146); local_mode / P_local: how the rank solves its own slab (THOMAS, or PDD / PPT with P_local
 * partitions per line).  The slab borrows slab_grid (destroy the slab first).  Plan-time work (global operator rows,
 * the cut slab operator, the rank's spikes, the rank-level reduced system) runs in CUDA kernels at creation.
 *
 * One sweep = three calls, all asynchronous on `stream`, all DEVICE buffers, 16-byte aligned:
 *   tdx_slab_eliminate  field_inout [slab] d -> xt = A_r^-1 d in place (Alg.1 steps 2-3) and iface_out[2][plane] =
 *                       (row 0, row n_loc-1) of xt; plane = the slab's other two extents (x fastest).
 *   (caller)            exchange: PDD -- send iface_out[0] to rank-1 and iface_out[1] to rank+1 (steps 4, 6);
 *                       PPT -- all-gather every rank's iface_out into [nranks][2][plane] (L156, L174).
 *   tdx_slab_correct    iface_own = this rank's iface_out; iface_nbr = PDD: [2][plane] = (xt_last of rank-1, xt_first
 *                       of rank+1), entries of a missing neighbour are not read; PPT: the gathered [nranks][2][plane].
 *                       Solves the interface unknowns per line (step 5 / Eq.(7)) and applies Eq.(8) (step 7) in place.
 * tdx_slab_dropped_bound: max |v_last|, |w_first| over interior ranks, the entries PDD across ranks deletes (L152). */
typedef struct tdx_slab tdx_slab_t;
tdx_status_t tdx_slab_create(tdx_grid_t* slab_grid, tdx_dir_t dir, int rank, int nranks, int n_global,
                             const double* faces_global, tdx_bc_t bc_global, double alpha, tdx_mode_t across,
                             tdx_mode_t local_mode, int P_local, tdx_slab_t** out);
tdx_status_t tdx_slab_destroy(tdx_slab_t* slab);
tdx_status_t tdx_slab_eliminate(tdx_slab_t* slab, double* field_inout, double* iface_out, void* stream);
tdx_status_t tdx_slab_correct(tdx_slab_t* slab, double* field_inout, const double* iface_own, const double* iface_nbr,
                              void* stream);
tdx_status_t tdx_slab_dropped_bound(tdx_slab_t* slab, double* out);

/* Batched tridiagonal solve with PER-LINE coefficients and diagonal pivoting ("a parallel tridiagonal
 * solver with diagonal pivoting is used [3]") -- for systems whose dominance the caller does not vouch for.
 * a, b, c: DEVICE, nx*ny*nz doubles each, laid out like the field: row j of a line holds a = coupling to row j-1,
 * b = diagonal, c = coupling to row j+1; a of a line's first row and c of its last row are not read by
 * tdx_general_solve and are the periodic corner couplings for tdx_general_cyclic_solve (a of row 0 couples it to row
 * n-1, c of row n-1 to row 0; n >= 3).  pivoting != 0: 1x1 / 2x2 diagonal pivots without row interchanges (criterion:
 * tdx_general.cuh); pivoting == 0: plain elimination on the same data (breaks down on a zero pivot: inf / nan in that line,
 * no error).  rhs_inout: DEVICE, in place; the coefficient arrays are not modified.  dir = x, y or z.
 * Two methods (tdx_general.cuh).  PARTITION: Eq.(5)-(8) with the pivoted elimination inside every 8-row partition, spikes and
 * reduced system on the fly, one pass over HBM (40 B per value); the result of every line is checked (componentwise
 * backward error of the line's equations) before it is stored, and a line that fails -- a numerically singular partition
 * block; the line itself may be regular -- is solved instead, in the same call, by the other method;
 * tdx_general_fallback_count says how many lines of the grid's last general solve that were (it synchronises).
 * With pivoting != 0 the partition pass runs OPTIMISTICALLY with plain elimination: a line is accepted when the LU factors of
 * all its blocks are componentwise stable (|L||U| <= 4|A|: true for row- or column-dominant rows) and the spikes stay <= 1, or
 * when it passes the backward-error check; every other line is re-solved WITH the diagonal pivots by the LINES method.  The flag
 * TDX_GENERAL_PIVOT_PARTITIONS keeps the pivots inside the partitions instead (fewer re-solved lines on non-dominant
 * systems, slower on dominant ones).
 * LINES: one thread per line, diagonal pivoting over the whole line, two passes over HBM (about 82 B per value).
 * Default: PARTITION wherever it applies (it measured faster in every direction on dominant systems) -- except
 * that a pivoting solve first samples 32768 rows ON THE DEVICE (no host synchronisation; the same choice for
 * the same input): where more than a quarter of them are not diagonally dominant, most lines would be re-solved anyway
 * and LINES runs on every line straight away (tdx_general_fallback_count then reports every line).  OR the flags below
 * into `pivoting` to force a method.  Periodic lines, and lines of fewer than 4 or more than 4096 rows, always take LINES.
 * work: DEVICE scratch, caller-owned, 8-byte aligned: 9*nx*ny*nz + 8 bytes (tdx_general_solve), 25*nx*ny*nz + 24 bytes
 * (tdx_general_cyclic_solve).  A singular line yields inf / nan in that line.  Asynchronous on `stream`.       */
#define TDX_GENERAL_PIVOT 1
#define TDX_GENERAL_FORCE_PARTITION 16
#define TDX_GENERAL_FORCE_LINES 32
#define TDX_GENERAL_PIVOT_PARTITIONS 64   /* PARTITION method: keep the 1x1 / 2x2 pivots inside the partitions (see below) */
tdx_status_t tdx_general_solve(tdx_grid_t* grid, tdx_dir_t dir, int pivoting, const double* a, const double* b,
                               const double* c, double* rhs_inout, void* work, void* stream);
tdx_status_t tdx_general_cyclic_solve(tdx_grid_t* grid, tdx_dir_t dir, int pivoting, const double* a, const double* b,
                                      const double* c, double* rhs_inout, void* work, void* stream);
tdx_status_t tdx_general_fallback_count(tdx_grid_t* grid, long long* out);

/* A solve that ALLOCATES NOTHING, for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid it): the Poisson y-solves (delta2_y - kx2[i] - kz2[m]) phi = rhs of
 * tdx_helmholtz_wavenumber_solve in mode THOMAS with per-line shifts (same kernel, same
 * arithmetic, same pinning of lambda == 0 lines), with two differences: kx2_dev (nx doubles) and kz2_dev (nm doubles) are
 * DEVICE arrays the caller owns (no upload, no cache), and the kernel's scratch (the scaled super-diagonal of every line,
 * nx*ny*nm doubles) is a static device array inside the library instead of a workspace the grid allocates.
 * Limit: nx*ny*nm <= TDX_STATIC_SCRATCH_DOUBLES (2 359 296 doubles = 18 MiB, held by every GPU that loads the library
 * until the process exits; config 2, 256 x 128 x 65 modes, fits); larger sizes return TDX_ERR_UNSUPPORTED and launch nothing.
 * The call makes no cudaMalloc / cudaFree and calls no allocating routine; the grid must exist already (its metric tables
 * are allocated by tdx_grid_create).  Negative or NaN wavenumbers cannot be checked here (they are on the device).
 * EVERY call on a device shares the one array: calls that overlap on the GPU (two streams, two host threads, two grids)
 * RACE -- order them on one stream or with events.  The array keeps the last call's contents; nothing in it needs to be
 * zero at entry (every entry is written before it is read).  rhs_inout: DEVICE, complex128 [nm][ny][nx], in place.
 * Asynchronous on `stream`.  tdx_static_scratch_setup(device) resolves the array's device address
 * (cudaGetSymbolAddress, once per device) ahead of time -- call it before a graph capture begins; otherwise the first
 * solve on a device does it.                                                                                      */
#define TDX_STATIC_SCRATCH_DOUBLES 2359296
tdx_status_t tdx_static_scratch_setup(int device);
tdx_status_t tdx_helmholtz_thomas_lines_static(tdx_grid_t* grid, int nm, const double* kx2_dev, const double* kz2_dev,
                                               double* rhs_inout, void* stream);

/* Batched cyclic tridiagonal solve along dir with caller-given coefficients shared by every line:
 * a, b, c: HOST arrays of n_dir doubles; a[0] couples row 0 to row n-1 and c[n-1] couples row n-1 to row 0.
 * Closure as for tdx_adi_sweep on a periodic direction (Sherman-Morrison with gamma = -b[0] for THOMAS, cyclic
 * reduced system for PDD / PPT).  rhs_inout: DEVICE, nx*ny*nz doubles. */
tdx_status_t tdx_cyclic_solve(tdx_grid_t* grid, tdx_dir_t dir, tdx_mode_t mode, int P,
                              const double* a, const double* b, const double* c,
                              double* rhs_inout, void* stream);

/* Same operations on HOST buffers: copy in, solve on the device, copy out, synchronous (returns when the result
 * is in host memory).  These are the end-to-end calls bench.py times for its "e2e" figure.
 * tdx_adi_step_host runs the x, y and z sweeps back to back on one upload.                               */
tdx_status_t tdx_adi_sweep_host(tdx_grid_t* grid, tdx_dir_t dir, tdx_mode_t mode, int P,
                                double alpha, double* host_rhs_inout);
tdx_status_t tdx_adi_step_host(tdx_grid_t* grid, tdx_mode_t mode, int Px, int Py, int Pz,
                               double alpha, double* host_rhs_inout);
tdx_status_t tdx_helmholtz_wavenumber_solve_host(tdx_grid_t* grid, tdx_mode_t mode, int P,
                                                 int nm, const double* kx2, const double* kz2,
                                                 double* host_rhs_inout);

/* One whole step on HOST buffers, pipelined: x, y and z sweeps of host_field (nx*ny*nz doubles; NULL skips it) and the
 * nm Helmholtz y-solves of host_helm (complex128 [nm][ny][nx]; NULL skips it).  The buffers travel in slabs over three
 * streams (upload, compute, download), so both PCIe directions are busy at once and the kernels hide behind the copies;
 * page-locked (pinned) host memory is needed for the overlap, pageable memory works but serialises.  Synchronous:
 * returns when both results are in host memory.  All plans are validated before the first copy. */
tdx_status_t tdx_step_host(tdx_grid_t* grid, tdx_mode_t mode, int Px, int Py, int Pz, double alpha, double* host_field,
                           int Ph, int nm, const double* kz2, double* host_helm);

/* The same step, enqueued only: returns as soon as its copies and kernels are in the three pipeline streams; the results are
 * in the host buffers once tdx_step_host_wait(grid, slot) has returned TDX_OK.  Two steps may be in flight, one per slot
 * (slot in {0, 1}; each slot has its own device staging, so the grid then holds two fields and two Helmholtz arrays).  One
 * call alone cannot beat three transfer times (the field must be up completely before any of it comes down -- the z sweep
 * needs every plane -- and the Helmholtz array shares the link with it); with two steps in flight the download of one
 * runs beside the upload of the next and the pair of PCIe directions stays busy: two transfer times per step.  The host
 * buffers of a slot must not be touched between the call and its wait; they must be page-locked for the call to be
 * asynchronous at all.  A slot that still holds a step returns TDX_ERR_INVALID_ARG; tdx_step_host is slot 0 followed by
 * its wait; the other *_host entry points wait for slot 0 first (they share its staging).  Calls on one grid from one
 * host thread at a time. */
tdx_status_t tdx_step_host_async(tdx_grid_t* grid, int slot, tdx_mode_t mode, int Px, int Py, int Pz, double alpha,
                                 double* host_field, int Ph, int nm, const double* kz2, double* host_helm);
tdx_status_t tdx_step_host_wait(tdx_grid_t* grid, int slot);

/* Diagnostics.  tdx_pdd_dropped_bound: max over interfaces of |v_last|, |w_first| for the ADI operator of
 * (dir, P, alpha) -- the entries PDD deletes from Z; the a-priori size of the PDD error.  */
tdx_status_t tdx_pdd_dropped_bound(tdx_grid_t* grid, tdx_dir_t dir, int P, double alpha, double* out);
/* The last PDD / PPT sweep kernel this host thread launched: name with template arguments and launch shape, e.g.
 * "k_strided<32,2,0,0,255,1> grid=(296,1,1) block=(8,16,1)" ("" before the first).  Thread-local, static storage.
 * bench.py keys the committed ncu captures (profiles/) by it: a changed kernel or launch shape invalidates them.  */
const char*  tdx_last_launch(void);
/* Number of kernels this library has launched on this process so far (all grids). */
long long    tdx_kernel_launch_count(void);
const char*  tdx_status_string(tdx_status_t status);
const char*  tdx_last_error(void);                  /* thread-local, static storage; "" when none          */
const char*  tdx_version(void);

#ifdef __cplusplus
}
#endif
#endif /* TDX_H */
