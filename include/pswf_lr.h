/* pswf_lr.h -- C ABI of the B200-native PSWF-LR reciprocal-space library.
 *
 * What it computes (arxiv/paper_2606_06617; line numbers refer to /root/reference/PAPER.md):
 * the reciprocal-space part of the PSWF-mollified inverse-power energy, Eq. (5),
 *
 *     E = 1/(2V) sum_a sum_{k != 0} Phi^_{p_a}(k) |rho_a(k)|^2 + sum_a E_0^{(p_a)},
 *     rho_a(k) = sum_j q_j^a exp(i k.r_j)                                   Eq. (6)
 *
 * for several channels a (latent charges q^a, exponent p_a in 1..6, 8 or 10), by the gridded algorithm of
 * (i) spread with the separable PSWF window, Eq. (20)-(21),(24); (ii) batched
 * forward 3-D FFT; (iii) diagonal scaling by Phi^_p(k)/W^(k)^2, Eq. (22),(25), with Phi^_p from
 * Eq. (14) / SI Theorem 1 (S47)-(S52) and the k = 0 constants of Eq. (17)-(19) / (S73),(S75),(S78),
 * (S79); (iv) Fourier-space reduction to E, Eq. (26); then -- as BASELINE.json's north_star asks,
 * and as the automatic-differentiation backward of (i)-(iv) does -- an inverse
 * FFT and a gather with the window and its derivative, giving per-atom potentials
 * phi_i^a = dE/dq_i^a and forces F_i = -dE/dr_i (q fixed).
 * pswf_lr_execute computes exactly that (no self term, no real-space term: the hot path).  The rows
 * SURVEY.md §8(f) ranks next are separate entry points: pswf_lr_execute_real (real-space complement
 * and self term, completing (S65)), pswf_lr_set_virial / pswf_lr_virial, pswf_lr_suggest_parameters.
 *
 * All kernels are CUDA for sm_100a; the 3-D FFTs are cuFFT.  There is no CPU fallback: every
 * call fails with PSWF_LR_ERR_CUDA when no device is usable.
 *
 * Conventions
 *   - Orthorhombic periodic box (Lx,Ly,Lz), k = 2 pi (mx/Lx, my/Ly, mz/Lz).
 *   - Lengths in Angstrom, energies in q^2 / A^p (Eq. (2) carries no prefactor).
 *   - "real" is float when the plan's precision is PSWF_LR_F32 and double for PSWF_LR_F64.
 *   - Every function returns 0 on success or a negative pswf_lr_status; no exception crosses
 *     the ABI.  pswf_lr_error_string() names a code.
 *   - A plan is bound to the CUDA device current at creation and owns every workspace, table
 *     and cuFFT plan; calls made while another device is current switch to the plan's device and
 *     restore the caller's afterwards.  One plan must not be executed from two streams at once.
 */
#ifndef PSWF_LR_H
#define PSWF_LR_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pswf_lr_plan pswf_lr_plan; /* opaque */

typedef enum {
  PSWF_LR_OK = 0,
  PSWF_LR_ERR_INVALID_ARG = -1,          /* null pointer, non-positive size, w out of range ...   */
  PSWF_LR_ERR_UNSUPPORTED_EXPONENT = -2, /* p not in {1..6, 8, 10} (SI Section 6)  */
  PSWF_LR_ERR_GRID_TOO_COARSE = -3,      /* h > pi r_c / c (Eq. (29)), w > M_d, or the window      */
                                         /* transform would be used outside its band              */
  PSWF_LR_ERR_ALLOC = -4,
  PSWF_LR_ERR_CUDA = -5,
  PSWF_LR_ERR_CUFFT = -6,
  PSWF_LR_ERR_BUSY = -7,                 /* host submissions in flight: pswf_lr_wait_host first    */
  PSWF_LR_ERR_TOO_LARGE = -8             /* size beyond the static scratch of a no-allocation call  */
} pswf_lr_status;

enum { PSWF_LR_F32 = 0, PSWF_LR_F64 = 1 };

/* Optional plan parameters; zero-initialise and set what you need (0 = default). */
typedef struct {
  double r_c;       /* mollifier cutoff r_c (A), Eq. (3),(13).  Default: c * max_d(h_d) / (0.5 pi),    */
                    /* i.e. eta = 0.5 in Eq. (29) (reading R2).                               */
  double c_window;  /* PSWF bandwidth of the spreading window (reading R3: separate from c).           */
                    /* Default: w * (3.55 - 1.55 eta), eta = c * max_d(h_d) / (pi r_c).                 */
  int precision;    /* PSWF_LR_F32 (default) or PSWF_LR_F64: type of pos, q, phi, F and the grids.     */
  int max_atoms;    /* capacity hint; buffers grow on demand.                                          */
  int zero_mode;    /* 0: the paper's k = 0 conventions (S73)/(S75)/(S78)/(S79), E_IB = 0 (default);   */
                    /* 1: drop the k = 0 mode.                                                          */
  int kernel_path;  /* 0: fastest available kernels (default); 1: simple reference kernels            */
                    /* (one warp per atom, global atomics) -- same arithmetic, for cross-checks.        */
  double poly_eps;  /* tolerance of the Horner tables.  Default 1e-7 (f32), 1e-12 (f64) */
  int host_only;    /* 1: build the host-side tables only (no device is touched); such a plan serves    */
                    /* pswf_lr_get_info / pswf_lr_eval_window / pswf_lr_eval_kernel and every compute    */
                    /* call on it fails with PSWF_LR_ERR_CUDA.  Not a CPU fallback.                      */
  int debug_spectrum; /* test hook: 1 keeps a dense copy of the scaled half spectrum for                 */
                    /* pswf_lr_debug_copy(what = 1) when the band-limited transform path is active      */
                    /* (that path never materialises the dense spectrum otherwise).                     */
} pswf_lr_opts;

/* Read-back of what the plan resolved (all host values). */
typedef struct {
  double r_c, c, c_window, eta;
  int w, precision, n_channels, n_distinct_p;
  int grid[3];
  int window_degree;     /* degree of the per-panel window polynomials                  */
  int kernel_degree;     /* degree of the per-panel polynomials for Phi^_p              */
  int kernel_panels;
  long long modes_in_ball;    /* half-spectrum modes with a non-zero multiplier          */
  long long workspace_bytes;  /* device memory owned by the plan                         */
  int fast_stencil;      /* 1: the cell-sorted fp32 spread / gather kernels run (fp32, w <= 8, M_d a     */
                         /*    multiple of 8 and >= 16, kernel_path = 0); 0: the one-warp-per-atom ones  */
  int band_limited_fft;  /* 1: z transforms + fused (x,y) transform / scale kernel (fp32, Mx and My      */
                         /*    powers of two <= 256, kernel_path = 0); 0: dense 3-D cuFFT                 */
  int band_kmax[3];      /* band-limited path: kept DFT indices |m_d| <= band_kmax[d]                    */
  long long own_kernel_launches; /* kernels of this library launched by the plan since creation (counted  */
  long long memsets;             /* at the launch sites), cudaMemsetAsync calls, and cuFFT executions      */
  long long cufft_execs;         /* (each a few cuFFT kernels; 0 on the band-limited path with pow-2 Mz)    */
  long long graph_replays;       /* evaluations replayed from a cached CUDA graph (their launches are      */
                                 /* included in the three counts above)                                    */
} pswf_lr_info;

/* Create a plan.  box[3]: edge lengths; grid[3]: M_x,M_y,M_z (each >= w, product < 2^31);
 * w: window width P in grid points (even, 2..16); c: mollifier bandwidth
 * (Eq. (28)), 2 <= c <= 60; exponents[n_channels]: p_a in 1..6 (Theorem 1) or 8, 10
 * (Theorem 2 / Corollary 1, (S55)-(S59)), repeats allowed.
 * Host pointers; nothing is retained.  Runs the host-side PSWF eigen-solve, fits the Horner
 * tables, builds cuFFT plans, allocates workspaces. */
int pswf_lr_plan_create(pswf_lr_plan** plan, const double box[3], const int grid[3], int w, double c,
                        const int* exponents, int n_channels);
int pswf_lr_plan_create_ex(pswf_lr_plan** plan, const double box[3], const int grid[3], int w,
                           double c, const int* exponents, int n_channels, const pswf_lr_opts* opts);

/* The same for a general (triclinic) periodic cell -- "positions, species and the cell tensor".
 * cell[9], row-major: row d is the lattice vector a_d (right-handed, det > 0); r = s h with fractional
 * s, k_m = 2 pi m h^-T, V = det h.  The grid has M_d points along a_d and the separable PSWF window
 * acts on the fractional coordinates; |a_d| / M_d takes the place of the grid spacing h_d in Eq. (29)
 * and in the defaults of r_c and c_window.  Positions, forces and the virial are Cartesian.  A diagonal
 * cell is the orthorhombic box of pswf_lr_plan_create_ex (same arithmetic).  pswf_lr_execute_real
 * takes the minimum image in fractional coordinates there (see its r_c condition). */
int pswf_lr_plan_create_cell(pswf_lr_plan** plan, const double cell[9], const int grid[3], int w,
                             double c, const int* exponents, int n_channels, const pswf_lr_opts* opts);

/* One evaluation, asynchronous on `stream` (a cudaStream_t; NULL = default stream).  No host
 * synchronisation and no host<->device copy happens inside (workspaces grow, with a sync, only
 * when n_atoms exceeds the capacity seen so far).
 *   pos  device, real[n_atoms][3]; any real coordinates (wrapped into the box internally)
 *   q    device, real[n_channels][n_atoms]
 *   E    device, double[1]: total energy, Eq. (26) (accumulated in double); may be NULL
 *   phi  device, real[n_channels][n_atoms], phi_i^a = dE/dq_i^a; may be NULL
 *   F    device, real[n_atoms][3], F_i = -dE/dr_i; may be NULL
 * Repeated calls with the same arguments (the same device buffers, as in an MD loop) are captured into a
 * CUDA graph on the second call and replayed afterwards; calls made while `stream` is itself being captured
 * launch plainly into the caller's capture.
 * Outputs are in the caller's atom order.  If phi and F are both NULL the inverse FFT and the
 * gather are skipped (the paper's energy-only path); with phi NULL and F given (an MD
 * step) the gather runs without the potential sums.  n_atoms = 0 is legal. */
int pswf_lr_execute(pswf_lr_plan* plan, int n_atoms, const void* pos, const void* q, void* E,
                    void* phi, void* F, void* stream);

/* Same evaluation with HOST buffers (pinned or pageable): copies pos and q to the device,
 * executes, copies E, phi, F back, all on `stream`, and synchronises the stream before
 * returning.  This is the end-to-end entry point bench.py times as "e2e". */
int pswf_lr_execute_host(pswf_lr_plan* plan, int n_atoms, const void* pos, const void* q, double* E,
                         void* phi, void* F, void* stream);

/* Pipelined form of pswf_lr_execute_host for streams of independent evaluations (batches of frames,
 * ensemble members, or an MD loop whose next positions do not wait for these forces): submit enqueues
 * the host->device copies, the evaluation and the device->host copies on three streams owned by the
 * plan and returns at once; at most THREE submissions may be in flight (three staging slots), a fourth
 * returns PSWF_LR_ERR_BUSY.  pswf_lr_wait_host blocks until the OLDEST outstanding submission has
 * delivered E, phi and F to its host buffers.  With pinned host buffers the copy-in of submission
 * k+1, the evaluation of k and the copy-out of k-1 overlap (PCIe is full duplex), so the sustained
 * cost per evaluation is max(copy-in, evaluation, copy-out) instead of their sum.  Host buffers must
 * stay valid and untouched until the matching wait returns.  Argument meaning as pswf_lr_execute_host
 * (there is no stream argument: the plan's own streams are used).  Not to be mixed with
 * pswf_lr_execute / pswf_lr_execute_host while submissions are in flight (PSWF_LR_ERR_BUSY). */
int pswf_lr_submit_host(pswf_lr_plan* plan, int n_atoms, const void* pos, const void* q, double* E,
                        void* phi, void* F);
int pswf_lr_wait_host(pswf_lr_plan* plan);

/* Real-space complement and self term: the part of the full inverse-power
 * energy (S65), that the reciprocal path above does not contain,
 *   E = 1/2 sum_a sum_{i != j, images} q_i^a q_j^a L_{p_a,r_c}(|r_ij|)  -  E_self,
 *   L_{p,r_c}(r) = r^-p - S_{p,r_c}(r) for r < r_c (SI Props. 2-7, (S17)-(S33)), 0 beyond;
 *   E_self = sum_a S_{p_a}(0) sum_i (q_i^a)^2 / (2 r_c^p_a)              (S66)-(S67).
 * Arguments as pswf_lr_execute; phi_i^a = dE/dq_i^a and F_i = -dE/dr_i of THIS part.  With
 * accumulate != 0 the results are ADDED to what E, phi and F already hold, so that
 *   pswf_lr_execute(...); pswf_lr_execute_real(..., 1, stream);
 * returns the complete energy, potentials and forces of (S65).  Asynchronous on `stream`; it re-sorts
 * the atoms (the plan's sort buffers are shared with pswf_lr_execute: same-stream use only).
 * Fails with PSWF_LR_ERR_GRID_TOO_COARSE when r_c is not below half the distance between opposite cell
 * faces in every lattice direction (L_d / 2 in an orthorhombic box; V / |a_e x a_f| / 2 in a general
 * cell): only the minimum image of a pair is visited. */
int pswf_lr_execute_real(pswf_lr_plan* plan, int n_atoms, const void* pos, const void* q, void* E,
                         void* phi, void* F, int accumulate, void* stream);

/* Virial ("forces and virials"): W_ab = -dE/d(eps_ab) under a
 * homogeneous strain of atoms and cell at fixed q and r_c.  After pswf_lr_set_virial(plan, 1) every
 * pswf_lr_execute accumulates the virial of the reciprocal energy in its scale kernel,
 *   W_ab = 1/2 sum_m D(m) |rho^(m)|^2 [delta_ab + (dD/dk)/(D |k|) k_a k_b]  (+ the k = 0 term),
 * the exact strain derivative of the gridded energy, and pswf_lr_execute_real adds (accumulate != 0) or
 * restarts (accumulate = 0) with the pair virial -1/2 sum_{i != j} q q L'(r) r_a r_b / r.
 * pswf_lr_virial copies it to a DEVICE buffer double[6] = xx, yy, zz, xy, xz, yz (async on stream).
 * Pressure: P = tr W / (3V) for this part of the energy. */
int pswf_lr_set_virial(pswf_lr_plan* plan, int enabled);
int pswf_lr_virial(pswf_lr_plan* plan, void* W, void* stream);

/* Per-channel energies of the most recent execute: device double[n_channels] (async on stream).
 * The paper reports per-component contributions. */
int pswf_lr_channel_energies(pswf_lr_plan* plan, void* E_channels, void* stream);

int pswf_lr_get_info(const pswf_lr_plan* plan, pswf_lr_info* info);

/* Stage timing with CUDA events recorded on the execute stream (for bench.py's roofline line).
 * Stages: 0 bin+sort, 1 spread, 2 forward FFT, 3 scale+reduce, 4 inverse FFT, 5 gather.
 * pswf_lr_stage_ms synchronises on the last event and returns, per stage, the mean milliseconds
 * over the executes since profiling was enabled (or last read), then resets the accumulation. */
enum { PSWF_LR_N_STAGES = 6 };
int pswf_lr_set_profiling(pswf_lr_plan* plan, int enabled);
int pswf_lr_stage_ms(pswf_lr_plan* plan, double ms[PSWF_LR_N_STAGES], int* n_executes);

/* Test hook: copy an intermediate of the most recent execute to a caller's DEVICE buffer.
 *   what = 0: real grid after spreading, real[n_channels][Mx][My][Mz]
 *   what = 1: scaled half-spectrum, 2*real[n_channels][Mx][My][Mz/2+1] (re,im interleaved)
 *   what = 2: potential grid after the inverse FFT, real[n_channels][Mx][My][Mz]
 * Only meaningful when the intermediate still exists (call right after execute; the real grid is
 * overwritten by the inverse FFT, so what = 0 needs an execute with phi = F = NULL). */
int pswf_lr_debug_copy(pswf_lr_plan* plan, int what, void* dst, void* stream);

/* Test hook: copy the cell starts of the most recent execute -- the exclusive scan of the atoms-per-cell
 * counts of step a0 (cell key = stencil cell (s_x, s_y, s_z), z fastest), with the
 * atom count in the last entry -- to a caller's DEVICE buffer int[Mx*My*Mz + 1]. */
int pswf_lr_debug_cell_starts(pswf_lr_plan* plan, int* dst, void* stream);

/* NO-ALLOCATION entry point, for callers that cannot call cudaMalloc (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid it): the exclusive scan of step a0 (cell counts -> cell starts, the
 * kernel the plans use) without a plan.  Its scratch -- the tile states of the single-pass scan -- lives in
 * a file-scope device array of the library (8200 bytes, held by every GPU that loads the library until the
 * process exits) instead of a cudaMalloc'd workspace.  The call performs no cudaMalloc / cudaFree and calls
 * no allocating library routine.
 *   counts: DEVICE pointer (current device), int[n + 1], 16-byte aligned.  In place: on return (stream
 *           order) counts[i] = counts_in[0] + ... + counts_in[i-1] for 0 <= i <= n, i.e. counts[n] = total
 *           (what counts[n] held on entry is ignored).  The total must fit in an int.
 *   n:      0 <= n <= PSWF_LR_SCAN_STATIC_MAX (2^24: a 256^3 grid); beyond it PSWF_LR_ERR_TOO_LARGE and
 *           nothing is launched.  NULL or misaligned counts, n < 0: PSWF_LR_ERR_INVALID_ARG.
 * Asynchronous on `stream`; no host synchronisation.  The scratch is SHARED by all calls of the process on
 * that GPU and keeps the previous call's contents (the call clears what it uses first): calls that overlap
 * on the GPU -- two streams, two host threads -- race; serialise them.  The first call on a device resolves
 * the array's device address (cudaGetSymbolAddress): make it once before capturing a graph. */
enum { PSWF_LR_SCAN_STATIC_MAX = 1 << 24 };
int pswf_lr_exclusive_scan_static(int* counts, int n, void* stream);

/* Host-side evaluation of the plan's fitted tables (tests compare them with the oracle):
 *   window:  W(z) and dW/dz for z in [-1,1) from the panel polynomials
 *   kernel:  Phi^_p(k) as the scale kernel evaluates it (k in 1/A) */
int pswf_lr_eval_window(const pswf_lr_plan* plan, int n, const double* z, double* W, double* dW);
int pswf_lr_eval_kernel(const pswf_lr_plan* plan, int p, int n, const double* k, double* Phi);
/*   real:    L_{p,r_c}(r) and dL/dr (r in A) from the numerator polynomials; S_p(0) of (S67) */
int pswf_lr_eval_real(const pswf_lr_plan* plan, int p, int n, const double* r, double* L, double* dL);
int pswf_lr_self_coefficient(const pswf_lr_plan* plan, int p, double* S0);

/* Parameter selection from a target tolerance (Eq. (27)-(29)).
 * Host-only, no plan needed.  eps_tot is split evenly, eps_band = eps_grid = eps_spread = eps_tot / 3:
 *   c    = ln(1 / eps_band)                                            Eq. (28)
 *   h   <= eta pi r_c / c with eta = 0.5 (reading R2), M_d = ceil(L_d / h) rounded up to a
 *          multiple of 8 (the fast kernels' granularity)               Eq. (29)
 *   w    = the smallest even window width in 4..16 whose spreading error estimate
 *          10^(0.46 - 0.85 w) (relative force error of the gridded scheme against the direct k-sum
 *          at eta = 0.5 and the default window bandwidth, fitted to the measured w = 6, 8, 12, 16
 *          values of DESIGN.md / SURVEY.md §8(c)) is <= eps_spread.
 * Returns PSWF_LR_ERR_INVALID_ARG for eps_tot outside [1e-13, 0.3] or non-positive box / r_c. */
int pswf_lr_suggest_parameters(const double box[3], double eps_tot, double r_c, int grid[3], int* w, double* c);

int pswf_lr_destroy(pswf_lr_plan* plan);
const char* pswf_lr_error_string(int code);
const char* pswf_lr_version(void);

#ifdef __cplusplus
}
#endif
#endif /* PSWF_LR_H */
