/*
 * dg.h — C ABI of libdg: the per-cell exponential drag update for a gas + N dust fluids (arXiv 2509.25347) on
 * NVIDIA B200 (sm_100a).  PAPER.md below is the extracted text of the paper; citations are PAPER.md:<line>.
 *
 * What the library computes, per cell and independently of every other cell (footnote 1):
 *     p_out[comp] = exp(dt * Omega) * p_in[comp],   comp = x, y, z                    (Eq. 18)
 * where Omega is the (N+1) x (N+1) drag matrix of Eq. 17 built from that cell's
 *     eps_i = rho_d,i / rho_g (Eq. 14)   and   alpha_i = 1 / t_s,i (Eq. 15),
 * and exp() is evaluated by Taylor-based scaling and squaring (Sect. 2.3; Alg. 6):
 * a norm-based choice of (m, s) from the thresholds of Table B.1, the degree-m Taylor polynomial
 * of A / 2^s (Eq. 19), then s squarings (Eq. 23-24).  Species index 0 is the gas.
 *
 * ---------------------------------------------------------------------------------------------------------------
 * Layouts.  Structure of arrays, fp64, cell index c fastest (0 <= c < ncells), n = N + 1, 1 <= N <= DG_NMAX:
 *     rho_g [ncells]             gas density                                  > 0
 *     rho_d [N][ncells]          dust densities                               >= 0
 *     t_s   [N][ncells]          stopping times                               > 0
 *     p     [3][n][ncells]       momenta (component, species, cell)           Eq. 13
 *     A, E  [n*n][ncells]        matrices, element r*n + col; row r = destination species, col = source species
 *     s_out [ncells]             int32, the scaling exponent s chosen in each cell
 * "Device pointer" = memory the GPU can address (cudaMalloc / a torch CUDA tensor's data_ptr()).
 * "Host pointer"   = ordinary host memory; page-locked (pinned) memory makes the copies asynchronous.
 *
 * Ownership.  The library owns no caller-visible memory and keeps no global state that affects results.  All
 * buffers are caller-allocated and caller-freed.  The dg_* device entry points allocate nothing and use no
 * workspace.  dg_drag_update_host keeps a private device staging area that dg_host_release() frees;
 * dg_drag_update_host_static stages in a fixed array inside the library image instead and allocates nothing.
 *
 * Streams and asynchrony.  `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Device
 * entry points only enqueue work and return; they never synchronise.  They are re-entrant and may be called
 * concurrently on different streams.
 *
 * Reproducibility.  For a fixed build and GPU the same call (same pointers' cell ranges, same ncells) gives the same
 * bits, run to run.  A cell's VALUE never depends on other cells beyond rounding: every cell agrees with the exact
 * result to the documented tolerance whatever its neighbours hold.  Its BITS may: the kernels pick the Taylor degree m
 * (any Table B.1 row is admissible for any cell) once per group of cells that share a warp — 32 cells of similar
 * stiffness out of a tile of 128 or 256 consecutive cells (tiles start at multiples of their size from cell 0) — so
 * computing the same cell as part of a different sub-range of the arrays (an offset that is not a multiple of 2048
 * cells, or another ncells where that cuts a tile short) may change its result at O(u).
 * dg_drag_update_host cuts its chunks so that it stays bit-identical to one dg_drag_update over all cells.
 *
 * Errors.  Every entry point returns a dg_status; nothing throws or aborts across the ABI:
 *     DG_ENULL   a required pointer is NULL (checked only when ncells > 0)
 *     DG_ERANGE  N outside [1, DG_NMAX] or ncells < 0
 *     DG_EALIGN  a pointer is not 8-byte aligned (fp64 arrays; 4-byte for the int32 arrays).  8 bytes is all that is
 *                required; 16-byte aligned base pointers with an even ncells let the kernels move whole rows of a tile
 *                per bulk copy (or two cells per copy) instead of one cell per copy — same results, faster
 *     DG_EINVAL  dt negative or not finite, or another scalar argument outside its documented range
 *     DG_ECUDA   the CUDA runtime reported an error (cudaGetLastError after the launch, or a failed copy/alloc);
 *                dg_last_cuda_error() returns its text
 *     DG_ECAPACITY  dg_drag_update_host_static only: ncells exceeds what its fixed staging array holds for this N
 * ncells == 0 is DG_OK and a no-op.
 *
 * Pre-conditions that are NOT checked on the device (PAPER.md is silent; they are what Eq. 14-15 need):
 * rho_g > 0, rho_d >= 0, t_s > 0, everything finite, rho_d / rho_g <= 1e200.  A cell that violates them yields
 * non-finite or meaningless output in that cell only.  dt = 0 returns p_out == p_in bit for bit.
 * rho_d,i = 0 is allowed: species i then receives nothing from the gas (column-0 entry i of Eq. 17 is zero).
 */
#ifndef DG_H
#define DG_H

#ifdef __cplusplus
extern "C" {
#endif

#define DG_NMAX 16
#define DG_VERSION 100 /* 0.1.0 */

typedef enum {
    DG_OK = 0, DG_EINVAL = 1, DG_ENULL = 2, DG_EALIGN = 3, DG_ERANGE = 4, DG_ECUDA = 5,
    DG_ECAPACITY = 6 /* dg_drag_update_host_static only: the cells do not fit its fixed staging array */
} dg_status;

/* ---- stage a1: assemble A = dt * Omega  (Eq. 14, 15, 17) ---------------------------------
 * in : rho_g, rho_d, t_s (device), dt.   out: A [n*n][ncells] (device), dense, including the structural zeros.
 * Off-diagonals: A[0][i] = dt/t_s,i, A[i][0] = (rho_d,i/rho_g) * dt/t_s,i.  Each diagonal entry is minus the sum
 * of the off-diagonal entries of its column (columns of Eq. 17 sum to zero: total momentum). */
dg_status dg_drag_matrix_build(const double* rho_g, const double* rho_d, const double* t_s, double dt, int N,
                               long long ncells, double* A, void* stream);

/* ---- stages a2-a4: E = exp(A) by scaling and squaring  (Sect. 2.3, Alg. 6, Table B.1) -----------------------
 * in : A [n*n][ncells] (device) — MUST be a drag matrix of Eq. 17 as dg_drag_matrix_build writes it: only the
 *      off-diagonal entries of row 0 and column 0 are read (A[0][i] >= 0, A[i][0] >= 0); the stored diagonal and
 *      the structural zeros are ignored and the diagonal is re-derived from the zero-column-sum property.  This is
 *      not a general-purpose expm.
 * out: E [n*n][ncells] (device), may alias A.  Entries are in [0,1] and every column sums to 1 to rounding.
 *      s_out (device, int32 [ncells], nullable): the scaling exponent chosen per cell (number of squarings). */
dg_status dg_expm_scale_square(const double* A, int N, long long ncells, double* E, int* s_out, void* stream);

/* ---- stage a5: p_out[comp] = E * p_in[comp] for the three components  (Eq. 18) ----------------
 * in : E [n*n][ncells], p_in [3][n][ncells] (device).   out: p_out [3][n][ncells] (device), may alias p_in. */
dg_status dg_drag_apply(const double* E, const double* p_in, int N, long long ncells, double* p_out, void* stream);

/* ---- fused a1..a5 in one kernel; no matrix ever reaches HBM.  This is the timed path. -----------------------
 * in : rho_g, rho_d, t_s, p_in (device), dt.   out: p_out (device), may alias p_in.
 * HBM traffic per cell: 8*(8N+7) bytes. */
dg_status dg_drag_update(const double* rho_g, const double* rho_d, const double* t_s, double dt, const double* p_in,
                         int N, long long ncells, double* p_out, void* stream);

/* Same as dg_drag_update and additionally writes s_out[c] (device int32 [ncells], nullable) and m_out[c]
 * (device int32 [ncells], nullable): the scaling exponent and Taylor degree chosen in each cell. */
dg_status dg_drag_update_ex(const double* rho_g, const double* rho_d, const double* t_s, double dt,
                            const double* p_in, int N, long long ncells, double* p_out, int* s_out, int* m_out,
                            void* stream);

/* ---- M drag steps in a row: the Dustybox driver  (Sect. 3.1, Eq. 26-30) ----------------------
 * Applies the fused update `nsteps` times with the same dt, densities and stopping times:
 *   p_out = exp(dt Omega)^nsteps p_in, every step computed from scratch by the fused kernel, as a hydro code calls it
 * once per time step (footnote 1).  nsteps launches on `stream`: the first reads p_in and writes
 * p_out, the rest run in place on p_out.  p_out may alias p_in.  nsteps = 0 copies p_in to p_out.
 * DG_EINVAL if nsteps < 0; otherwise the errors of dg_drag_update. */
dg_status dg_drag_update_steps(const double* rho_g, const double* rho_d, const double* t_s, double dt,
                               const double* p_in, int N, long long ncells, int nsteps, double* p_out, void* stream);

/* ---- first-order implicit RK1 drag step, O(N) closed form  (App. A.2, Eq. A.6-A.9) ----------
 * p_out[comp] = (I - dt Omega)^-1 p_in[comp] for the three components, Omega of Eq. 17: the backward-Euler solver the
 * paper uses as its speed reference (Fig. 6-7) and as the first-order accuracy reference (Fig. 2).  Not part of the
 * EXP path; same buffers, layouts, aliasing rule (p_out may alias p_in) and errors as dg_drag_update.
 * HBM traffic per cell: 8*(8N+7) bytes, O(N) flops. */
dg_status dg_drag_rk1(const double* rho_g, const double* rho_d, const double* t_s, double dt, const double* p_in,
                      int N, long long ncells, double* p_out, void* stream);

/* ---- drag update + gas energy with frictional heating  (Eq. 4 and Eq. 11) ----------------------
 * p_out as dg_drag_update, and the gas total energy E_g = |M_g|^2/(2 rho_g) + e after the drag step:
 *     E_out = E_in + [KE_g(p_out) - KE_g(p_in)] + w * [K(p_in) - K(p_out)],
 * K = |M_g|^2/(2 rho_g) + sum_i |M_d,i|^2/(2 rho_d,i) the total kinetic energy of the cell.  This is Eq. 4's drag part
 * integrated exactly along the exact momenta (the paper prints no discrete formula; reading R20): the first
 * bracket is the work of the drag force on the gas, the second the kinetic energy the drag dissipates, of which the
 * fraction w (0 = no frictional heating, 1 = all of it) is deposited into the gas.  With w = 1,
 * E_g + sum_i |M_d,i|^2/(2 rho_d,i) is conserved.  A species with rho_d,i = 0 carries no energy.
 * in : rho_g, rho_d, t_s, p_in, E_in [ncells] (device), dt, w.   out: p_out (may alias p_in), E_out [ncells] (may alias
 * E_in).  One launch on `stream` for every N (the sums are formed inside the update kernel).
 * DG_EINVAL if w is outside [0, 1]; otherwise the errors of dg_drag_update. */
dg_status dg_drag_update_energy(const double* rho_g, const double* rho_d, const double* t_s, double dt,
                                const double* p_in, const double* E_in, double w, int N, long long ncells,
                                double* p_out, double* E_out, void* stream);

/* ---- the fused update in SINGLE precision  (Eq. B.8 with u = 2^-24) -------------------------------
 * The same path a1..a5 with every array and every operation in fp32, and (m, s) chosen against the scaling thresholds
 * theta_m of Eq. B.4-B.8 recomputed for the unit round-off of IEEE single precision (the paper's Table B.1 is the
 * u = 2^-53 column; Eq. B.8 names 2^-24 as an alternative).  Layouts as above with float elements; pointers 4-byte
 * aligned (16-byte aligned arrays with ncells a multiple of 4 move whole tile rows per bulk copy: same results, faster);
 * p_out may alias p_in; s_out, m_out (int32 [ncells]) nullable.  Agrees with the exact result to about
 * (s + m + 8)(N + 2) 2^-24 max|p_in| per cell; total momentum to a few 2^-24. */
dg_status dg_drag_update_f32(const float* rho_g, const float* rho_d, const float* t_s, float dt, const float* p_in,
                             int N, long long ncells, float* p_out, int* s_out, int* m_out, void* stream);

/* Same as dg_drag_update_ex with the thread mapping forced (for measuring the mappings against each other; both
 * compute the same arithmetic and agree to rounding):
 *   DG_VARIANT_DEFAULT  the library's measured choice for this N (what dg_drag_update uses)
 *   DG_VARIANT_TPC      thread-per-cell: one thread owns a cell, packed symmetric matrices in registers; a warp takes
 *                       32 consecutive cells
 *   DG_VARIANT_WPC      warp-per-cell: one warp owns a cell, fp64 tensor-core (DMMA) tiles for the squarings
 *   DG_VARIANT_PPC      pair-per-cell: two lanes own a cell, the iterate in a shared-memory tile, cells sorted by
 *                       stiffness inside tiles of 128 cells before they are handed to the warps (default, N >= 13)
 *   DG_VARIANT_PAPER    NOT the same arithmetic: the paper's own scheme as printed — one thread per cell, dense
 *                       (N+1)x(N+1) fp64 matrices, Table B.1 row minimising Pi_m + s on ||A||_1 (Eq. B.11), Taylor
 *                       polynomial by Algorithm 7, plain squarings (Alg. 6).  A measured reference for the design
 *                       comparison; its error grows like 2^s u on stiff cells.
 *   DG_VARIANT_PAPER_ALG2   as DG_VARIANT_PAPER with (m, s) chosen by the paper's Algorithm 2 as printed
 *                       (the branch-reduced "first modification" of Sastre et al.)
 *   DG_VARIANT_PAPER_BOUND  as DG_VARIANT_PAPER_ALG2 plus the "second modification": the bound b_exp by Algorithm 8
 *                       and the evaluation with bound test by Algorithm 9; m_out then
 *                       reports the degree actually evaluated, m - q * (blocks the test dropped)
 *   DG_VARIANT_TPS      thread-per-cell over sorted tiles (default for N <= 12; DG_EINVAL above): a block stages a tile
 *                       of 128 or 256 consecutive cells in shared memory with bulk copies, counting-sorts it by
 *                       stiffness and hands its warps chunks of 32 cells that need about the same number of squarings
 * Any other value is DG_EINVAL. */
#define DG_VARIANT_DEFAULT 0
#define DG_VARIANT_TPC 1
#define DG_VARIANT_WPC 2
#define DG_VARIANT_PAPER 3
#define DG_VARIANT_PPC 4
#define DG_VARIANT_PAPER_ALG2 5
#define DG_VARIANT_PAPER_BOUND 6
#define DG_VARIANT_TPS 7
dg_status dg_drag_update_variant(const double* rho_g, const double* rho_d, const double* t_s, double dt,
                                 const double* p_in, int N, long long ncells, double* p_out, int* s_out, int* m_out,
                                 int variant, void* stream);

/* ---- the same update on HOST buffers (end-to-end path) -------------------------------------------------------
 * All array arguments are HOST pointers in the layouts above.  The call cuts the cells into chunks of
 * `chunk_cells` (0 = library default; rounded up to a multiple of 2048 cells so that the result is bit-identical
 * to one dg_drag_update launch over all cells), copies each chunk's inputs to a private device staging area, runs the
 * fused kernel and copies the result back, overlapping the three on internal streams; it returns after the last
 * copy has completed (it synchronises).  Page-locked host buffers make the copies truly asynchronous; pageable
 * buffers work but serialise.  p_out may alias p_in.  `device` is the CUDA device ordinal (-1 = current). */
dg_status dg_drag_update_host(const double* rho_g, const double* rho_d, const double* t_s, double dt,
                              const double* p_in, int N, long long ncells, double* p_out, long long chunk_cells,
                              int device);
/* Frees the staging area and streams of dg_drag_update_host (all devices).  Safe to call at any time. */
dg_status dg_host_release(void);
/* Test hook, not needed in normal use: lowers the largest row pitch (bytes) for which dg_drag_update_host uses one
 * strided 2-D copy per array; rows with a larger pitch are copied one by one (what happens by itself from
 * ncells >= 2^28).  0 restores the device's own limit.  Results do not depend on it.  DG_EINVAL if bytes < 0. */
dg_status dg_host_set_max_pitch(long long bytes);

/* ---- the same update on HOST buffers, for callers that cannot allocate device memory ---------------------------
 * dg_drag_update_host obtains its device staging area with cudaMalloc.  That rules it out for a caller whose own
 * memory pool has claimed the whole GPU at start-up (the request would fail), for a time-step loop that must not
 * stall (cudaMalloc / cudaFree synchronise the device), for a process held to a device-memory quota, and for a plug-in
 * whose host application forbids allocation after initialisation.  This entry point is for them: it makes no
 * cudaMalloc, cudaFree or any other allocating call, and creates no streams or events.  Its staging area is a fixed
 * array of DG_STATIC_STAGE_BYTES inside the library image, which every GPU that loads the library's module for this
 * entry point holds from that moment until the process exits, whether the entry point is called again or not.
 *
 * in : rho_g, rho_d, t_s, p_in (HOST, layouts above with row pitch ncells), dt.   out: p_out (HOST), may alias p_in.
 * Runs on the CURRENT device, entirely on `stream`: four host-to-device copies, the kernel dg_drag_update uses for
 * this N over all ncells at once, one device-to-host copy; then it waits for `stream`, so p_out is complete on return.
 * The result is bit-identical to dg_drag_update_host and to dg_drag_update on the same cells.
 *
 * Size limit.  A cell needs 8N + 7 doubles of staging (inputs, momenta in, momenta out), so
 *     ncells <= DG_STATIC_STAGE_BYTES / (8 * (8N + 7))     (279 620 cells at N = 1, 59 074 at N = 8, 31 068 at N = 16).
 * A larger ncells returns DG_ECAPACITY before any CUDA call is made; nothing is copied and p_out is untouched.  There
 * is no internal chunking: a caller with more cells compacts them into pieces of at most that many cells and calls once
 * per piece (pieces that are multiples of 2048 cells reproduce the bits of one launch over everything).
 *
 * First call.  The first call on each device resolves the array's device address (cudaGetSymbolAddress), which also
 * makes the CUDA runtime load the module and place the array on that device.  Make that first call during start-up:
 * before any stream capture is begun, and at a point where a one-off driver-side set-up cost is acceptable.
 *
 * Sharing.  There is ONE array per device, shared by every call in the process, and it keeps the previous call's
 * bytes.  That is harmless for a single caller — each call overwrites every value its kernel reads, and nothing needs
 * to start at zero, so nothing is cleared — but two calls whose GPU work can overlap (two host threads, whatever their
 * streams) race on the array and corrupt each other's results.  The library does not serialise them: the caller must.
 * Other errors as dg_drag_update_host. */
#define DG_STATIC_STAGE_BYTES 33554432 /* 32 MiB */
dg_status dg_drag_update_host_static(const double* rho_g, const double* rho_d, const double* t_s, double dt,
                                     const double* p_in, int N, long long ncells, double* p_out, void* stream);

/* ---- measurement helpers (used by bench.py; not on the data path) --------------------------------------------
 * dg_peak_kernel enqueues ONE launch of a microbenchmark kernel on `stream` and returns in *work the number of
 * flops (kinds 0-2; FMA = 2) or bytes (kind 3) that launch performs; the caller times it with events.
 *   kind 0: independent fp64 FMA chains (DFMA), all SMs        kind 1: fp64 tensor-core tiles (DMMA m8n8k4)
 *   kind 2: DFMA and DMMA interleaved in the same warps        kind 3: fp64 SoA copy (read + write bytes)
 * scratch: device buffer of at least scratch_bytes bytes (>= 1 MiB; kind 3 copies its first half to its second).
 * iters: loop trip count per thread (kinds 0-2). */
dg_status dg_peak_kernel(int kind, int iters, double* scratch, long long scratch_bytes, double* work, void* stream);

/* Number of kernels ONE call of dg_drag_update (or _ex, _variant, _f32, _rk1) enqueues for these arguments: 1, or 0
 * if ncells == 0 (dg_drag_update_energy likewise).  Not for the other entry points: dg_drag_update_steps enqueues
 * nsteps times as many, dg_drag_update_host one per chunk. */
int dg_launches_per_update(int N, long long ncells);
/* Human-readable description of the kernel variant dg_drag_update uses for N (static storage). */
const char* dg_variant_name(int N);

const char* dg_status_string(dg_status st); /* static storage */
const char* dg_last_cuda_error(void);       /* static storage; "" if none */
int dg_version(void);

#ifdef __cplusplus
}
#endif
#endif /* DG_H */
