/*
 * spray.h -- C-ABI of libspray_b200: the SPH particle-pair summation pass of SPRAY
 * (arxiv/paper_2604_20124) as hand-written CUDA for sm_100a, one GPU, fp64.
 *
 * Citations: "P:L<n>" = line n of the paper text; "A<n>" = reading n of DESIGN.md §3
 * (where the paper is silent, ambiguous or garbled).
 *
 * Conventions (all entry points)
 *   - return value: 0 = SPRAY_OK, < 0 = error (enum below).  No exception, exit or abort crosses the ABI.
 *     spray_last_error(ctx) returns a ctx-owned, NUL-terminated description of the last failure.
 *   - every array pointer is a DEVICE pointer owned by the caller (fp64 or u32/u64 as typed, contiguous,
 *     8-byte aligned, length n unless stated, CALLER ORDER = the order given to spray_build_cells).
 *     The library neither frees nor keeps them beyond the stream work the call enqueues.
 *     Output arrays must not alias inputs.  "nullable" outputs are skipped when NULL.
 *   - `stream` is a cudaStream_t passed as void* (e.g. torch.cuda.current_stream().cuda_stream).  Calls only
 *     ENQUEUE work on it and return; none synchronises except spray_check, spray_create and spray_destroy.
 *   - the ctx owns all scratch (sorted SoA copies, keys, permutation, cell tables, neighbour lists), sized at
 *     spray_create for n_max particles and ncell_max cells.  A ctx is bound to one device and is not
 *     thread-safe; use one ctx per stream.
 *   - inputs are not validated on the device: NaN or non-positive h, rho, E, kappa propagate as in the
 *     defining formulas.  Host-checkable errors (sizes, grid) are reported by the return code; device-side
 *     findings (h > declared h_max, position outside a periodic box, neighbour-list capacity exceeded)
 *     are latched into a sticky status word read by spray_check.
 *
 * Notation: x_ab = x_a - x_b, r = |x_ab|, q = r/h; grad_a W(x_ab,h) = F(r;h) x_ab / r with F = dW/dr (A4);
 *   V_b = m_b / rho_b.  Support radius is 2h for both kernels ("kappa = 2").
 *   N_gather(a) = { b : r^2 < 4 h_a^2 } (contains a);  N_sym(a) = { b != a : r^2 < 4 max(h_a,h_b)^2 } (A13:
 *   the mutual-neighbour set the paper's h' device produces).  r^2 = fma(dz,dz,fma(dy,dy,dx*dx)) with
 *   minimum-image dx in periodic dimensions (A12, A15); the predicates are evaluated in exactly this form.
 */
#ifndef SPRAY_H_
#define SPRAY_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct spray_ctx spray_ctx;

typedef enum {
    SPRAY_OK = 0,
    SPRAY_ERR_INVALID_ARG = -1,
    SPRAY_ERR_NOT_BUILT = -2,      /* a sweep was called before spray_build_cells succeeded */
    SPRAY_ERR_GRID = -3,           /* ncell_d < 1, prod ncell_d > ncell_max, hi <= lo, or periodic L_d < 3*(2*h_max) */
    SPRAY_ERR_CAPACITY = -4,       /* n > n_max */
    SPRAY_ERR_CUDA = -5,
    SPRAY_ERR_ALLOC = -6,
    SPRAY_ERR_NOT_IMPLEMENTED = -7
} spray_status_t;

/* sticky device-side status bits returned by spray_check */
enum {
    SPRAY_DEV_H_EXCEEDS_HMAX = 1,  /* some h_a > grid.h_max (search range may be incomplete) */
    SPRAY_DEV_OUTSIDE_BOX = 2,     /* a position outside [lo,hi) in a periodic dimension, or NaN */
    SPRAY_DEV_LIST_OVERFLOW = 4    /* neighbour-list storage exhausted (results of the tiled path invalid) */
};

typedef enum { SPRAY_KERNEL_CUBIC_SPLINE = 0, SPRAY_KERNEL_WENDLAND_C2 = 1 } spray_kernel_t;
typedef enum { SPRAY_FLD_SYMMETRIC = 0, SPRAY_FLD_GATHER = 1 } spray_fld_kernel_mode_t;       /* A17 */
typedef enum { SPRAY_FLD_UPDATE_LIMITER = 0, SPRAY_FLD_FROZEN = 1,
               /* FROZEN, called right after spray_hydro_rhs_limiter on this context with the same m, rho, E arrays and the mu array
                * that call wrote: the sorted operator records it left are reused and the per-call prologue (one pass over all
                * particles) is skipped; same results bit for bit.  SPRAY_ERR_INVALID_ARG if the context did anything else since. */
               SPRAY_FLD_FROZEN_CHAINED = 2 } spray_fld_limiter_mode_t; /* A18 */

/* Uniform cell grid (an INPUT, A14; "dimensions of these cells are ... determined based on the average
 * smoothing length ... during the initialization phase").  h_max is the caller-declared upper bound on h. */
typedef struct {
    double lo[3], hi[3];
    int32_t ncell[3];
    int32_t periodic[3];
    double h_max;
} spray_grid_t;

/* Library / build information: "spray-b200 <version> sm_100a". Static string. */
const char* spray_version(void);

/* Create a context on CUDA device `device` with scratch for n_max particles and ncell_max cells.
 * Host call; allocates device memory (SPRAY_ERR_ALLOC on failure). *out is set only on success. */
int spray_create(spray_ctx** out, int64_t n_max, int64_t ncell_max, int device);
/* Frees all scratch.  Synchronises the device. NULL is accepted. */
int spray_destroy(spray_ctx* ctx);
const char* spray_last_error(const spray_ctx* ctx);

/* Debug: synchronises `stream`, stores the sticky device status bits in *dev_status (nullable) and clears them.
 * Returns SPRAY_ERR_CUDA if any enqueued kernel faulted. */
int spray_check(spray_ctx* ctx, void* stream, uint32_t* dev_status);

/* Number of CUDA kernels this context has launched since spray_create (bench.py reports it as gpu_launches). */
int64_t spray_launch_count(const spray_ctx* ctx);

/* Select the pair-kernel implementation: 0 = reference kernels (one thread per particle walking the cell
 * table), 1 = tiled kernels (shared-memory staged neighbour cells + per-particle neighbour lists built
 * once per spray_build_cells).  Default 1 where available.  Both are CUDA; neither touches the host. */
int spray_set_path(spray_ctx* ctx, int path);

/* Debug/measurement: synchronises `stream`; *n_tiles = tiles of the tiled path built by the last spray_build_cells,
 * *n_fast = particles served by the tiled kernels (the rest, n - n_fast, by the general kernels),
 * *n_nonuniform = list-builder work units (half tiles) whose particles do not all share one h (they run the
 * variable-h pair bodies), *scratch_bytes = device memory the context holds (allocated at spray_create).
 * declined[k] = targets (k = 1: warps) the list builder left to the general kernels, by reason: 0 unused, 1 list pool
 * exhausted (per warp of 16 targets), 2 a list longer than 160 neighbours or more than 24 neighbours in one shared-memory
 * bank, 3 other (coincident particles, particle outside the tile's fp32 range).  With internal levels the counts are summed
 * over the levels.  All host pointers, all nullable. */
int spray_path_stats(spray_ctx* ctx, void* stream, int64_t* n_tiles, int64_t* n_fast, int64_t* n_nonuniform,
                     int64_t* scratch_bytes, int64_t* declined /* [4] */);

/* Internal levels of the tiled path, for particle sets whose smoothing lengths do not fit one grid (the search
 * range of a particle follows from the ratio of its smoothing length to the cell size, and neighbours are made mutual).
 * The tiled kernels need every mutual neighbour of a particle within one cell of the grid they work on; where the caller's
 * grid (an input, A14) does not give that -- cell edge below 2 h for some particles, or cells holding far more particles
 * than a tile can stage for others -- the library sorts the particles a second, third, ... time on grids of its own over
 * the same box: level k has ncell_d = floor(L_d / edges[k]) cells and serves the particles a with 2 hs_a (hs = symmetric
 * search length: max of h_a and the h of every particle that sees a) above the cell edge of level k - 1 and not above that
 * of level k; what no level can take (2 hs above the last edge, more than 160 neighbours in one part of a tile) stays with the
 * general kernels, so results are complete and identical either way.  edges: host, [nlevels], ascending, > 0 (a good
 * choice: a geometric sequence of ratio ~1.5 from 2 min(h) to 2 max(h)); ncell_max: host, [nlevels], cell capacity of each
 * level (>= prod floor(L_d / edges[k])).  Allocates the levels' scratch (synchronises the device; call it once, before
 * spray_build_cells); nlevels = 0 removes them.  Returns SPRAY_ERR_ALLOC when a level cannot be allocated (none is kept).
 * The cell table, the sort permutation and every output are those of the caller's grid regardless. */
int spray_set_levels(spray_ctx* ctx, int nlevels, const double* edges, const int64_t* ncell_max);

/* Measurement: device time of the three parts of the LAST spray_build_cells on this context, from CUDA events the call
 * records on its stream (no cost on the path): *ms_cells = keys, sort, cell table, reorder, per-cell h_max, symmetric
 * search length (a1-a4); *ms_tiles = coincidence marks, tile cutting, tile tables; *ms_lists = the neighbour-list
 * builder (k_build_lists).  The last two are 0 on path 0.  Synchronises on the build's last event.  Host pointers,
 * nullable. */
int spray_build_timing(spray_ctx* ctx, double* ms_cells, double* ms_tiles, double* ms_lists);

/* (a1)-(a4) NNPS: cell index per particle  c_d = floor((x_d - lo_d) * ncell_d / L_d) clamped,
 * key = (c_z*ncell_y + c_y)*ncell_x + c_x;  STABLE sort of (key, caller index);  cell_start[c] = #{key < c},
 * cell_end[c] = cell_start[c] + #{key = c};  sorted SoA copies of x, y, z, h;  per-cell max h;  per-particle
 * symmetric search length;  neighbour lists for the tiled path.
 * Stores `kernel` for the sweeps that follow.  x, y, z, h: device, [n], caller order, read only.
 * Errors: SPRAY_ERR_CAPACITY (n > n_max), SPRAY_ERR_GRID, SPRAY_ERR_INVALID_ARG (NULL, n < 0). n = 0 is valid. */
int spray_build_cells(spray_ctx* ctx, const spray_grid_t* grid, spray_kernel_t kernel, int64_t n,
                      const double* x, const double* y, const double* z, const double* h, void* stream);

/* (a1)-(a3) WITHOUT A CONTEXT AND WITHOUT ANY ALLOCATION: cell key, stable sort of (key, caller index) and the cell table of
 * P:L438, exactly as spray_build_cells computes them (same kernels and pass order: results are bit-identical to
 * spray_build_cells + spray_get_cell_table), for callers that cannot call cudaMalloc -- code under CUDA graph capture, tight
 * serving loops, harnesses that forbid it.  The call makes no cudaMalloc / cudaFree and uses no allocating library routine:
 * the sort's scratch (two key/index buffers, radix histograms, a status word) is a file-scope device array of
 * SPRAY_STATIC_SCRATCH_BYTES that every GPU loading the library holds until the process exits.
 *   grid: host (h_max is not used);  x, y, z: device, [n], read only;  outputs, all device, caller-allocated, must not alias
 *   the inputs: sorted_key[n], perm[n] (perm[i] = caller index of the particle in sorted slot i), cell_start[ncell],
 *   cell_end[ncell];  dev_status: device, one word, nullable: receives the SPRAY_DEV_* bits of this call (OUTSIDE_BOX).
 *   Works on the CURRENT device (cudaGetDevice), to which stream and pointers must belong.  Only enqueues.
 * Limits: n <= SPRAY_STATIC_NMAX (SPRAY_ERR_CAPACITY beyond, nothing is launched), prod ncell_d <= SPRAY_STATIC_NCELL_MAX
 * (SPRAY_ERR_GRID).  n = 0 is valid (empty cell table).  SPRAY_ERR_INVALID_ARG for NULL pointers / n < 0.
 * spray_static_last_error() returns the calling thread's description of its last failure of this call.
 * SHARED STATE: every call on a device uses the same array, which keeps the previous call's contents (the call clears what
 * must start at zero).  Two calls that overlap on the GPU -- different streams, or different host threads -- RACE on it
 * and give wrong results: serialise them (one stream, or events). */
#define SPRAY_STATIC_NMAX 262144
#define SPRAY_STATIC_NCELL_MAX 16777216
#define SPRAY_STATIC_SCRATCH_BYTES (4 * 1024 * 1024 + 128 * 1024)
int spray_cell_list_static(const spray_grid_t* grid, int64_t n, const double* x, const double* y, const double* z,
                           uint32_t* sorted_key, uint32_t* perm, uint32_t* cell_start, uint32_t* cell_end,
                           uint32_t* dev_status, void* stream);
const char* spray_static_last_error(void);

/* (a5) density by summation, eq. (35):  rho_a = sum_{b in N_gather(a)} m_b W(r_ab; h_a), self included (A11).
 * nnbr (nullable, u32[n]) = |N_gather(a)| - 1. */
int spray_density(spray_ctx* ctx, const double* m, double* rho, uint32_t* nnbr, void* stream);

/* (a6) hydro right-hand sides over N_sym(a) (pairs with r = 0 skipped, A11):
 *   momentum, eq. (11) P:L98 with the sign of eqs. (5), (19) (A3):
 *       a_a  = - sum_b m_b/(rho_a rho_b) [ p_a F(r;h_a) + p_b F(r;h_b) ] xhat_ab
 *   dissipation, eqs. (41), (43) P:L236-L242, applied for w = v_ab . xhat_ab < 0 (A6), vsig_s = alpha_s c_s + beta |w| (A8):
 *       a_a += sum_b (m_b/2) [ vsig_a F(r;h_a)/rho_a + vsig_b F(r;h_b)/rho_b ] w xhat_ab
 *   divergence sum, eq. (37):   divv_sum_a = D_a = sum_b V_b w F(r;h_a)      (d rho/dt = rho D;  div v = -D)
 *   energy, eq. (17) first term P:L129 + eq. (42) P:L238 (A7):
 *       dudt_a = (p_a/rho_a) D_a - (1/rho_a) sum_b (m_b vsig_a / 2) w^2 F(r;h_a)
 * Inputs [n] caller order; beta = 2 in the paper.  divv_sum nullable. */
int spray_hydro_rhs(spray_ctx* ctx, const double* m, const double* rho, const double* p, const double* cs,
                    const double* vx, const double* vy, const double* vz, const double* alpha, double beta,
                    double* ax, double* ay, double* az, double* dudt, double* divv_sum, void* stream);

/* (a6) + (a7) in one sweep: the hydro right-hand sides of spray_hydro_rhs AND the flux-limiter pre-sweep of spray_fld_apply
 * (P:L275 with grad E by eq. (9), phi = 1:  gradE_a = sum_{b in N_gather(a)} V_b (E_b - E_a) gradW(x_ab, h_a),  R_a = |gradE_a| /
 * (rho_a kappa_a E_a),  lambda_a = 1/sqrt(9 + R_a^2),  mu_a = c lambda_a / (rho_a kappa_a)).  Both sums need rho and nothing of each
 * other, and where h is uniform over a tile N_gather = N_sym, so the limiter's pair term reuses x_ab, 1/r and F/r of the hydro
 * pair: results are BITWISE those of spray_hydro_rhs followed by spray_fld_apply(SPRAY_FLD_UPDATE_LIMITER)'s mu / gradE (same
 * pair terms, same summation order; tiles with variable h and the particles of the general path run the two sweeps one after
 * the other inside this call).  Follow it with spray_fld_apply(..., SPRAY_FLD_FROZEN, mu, ...) for y, Lambda, Gamma.
 * Inputs [n] caller order as in the two calls; outputs ax, ay, az, dudt, mu [n]; divv_sum [n] and gradE [3n] nullable.
 * Errors: SPRAY_ERR_INVALID_ARG (NULL). */
int spray_hydro_rhs_limiter(spray_ctx* ctx, const double* m, const double* rho, const double* p, const double* cs,
                            const double* vx, const double* vy, const double* vz, const double* alpha, double beta,
                            const double* E, const double* kappa, double c_light,
                            double* ax, double* ay, double* az, double* dudt, double* divv_sum, double* mu, double* gradE, void* stream);

/* (a7)+(a8) matrix-free apply of the SPH flux-limited-diffusion operator.
 *   limiter pre-sweep (UPDATE_LIMITER only), P:L275 with grad E by eq. (9), phi = 1 (A19), over N_gather(a)\{a}:
 *       gradE_a = sum_b V_b (E_b - E_a) F(r;h_a) xhat_ab;   R = |gradE|/(rho kappa E);
 *       lambda = 1/sqrt(9 + R^2) (Larsen, k = 2, A20);   mu = c_light * lambda / (rho kappa)   -> written to mu[]
 *   apply, eq. (47) first term P:L270 / eqs. (51)-(52) P:L283-L286 on the Laplacian form eq. (16) P:L125:
 *       c_ab = V_b * 4 mu_a mu_b/(mu_a + mu_b) * Fbar/r
 *       Fbar = (F(r;h_a)+F(r;h_b))/2 over N_sym(a)  [SPRAY_FLD_SYMMETRIC, A17]   or  F(r;h_a) over N_gather(a)\{a}  [SPRAY_FLD_GATHER]
 *       y_a = sum_b c_ab (E_a - E_b) (difference form);  diag_a = Lambda_a = sum_b c_ab;  offd_a = Gamma_a = - sum_b c_ab E_b
 * FROZEN: mu[] is read as given (the linear operator an implicit solve applies every iteration).
 * kappa may be NULL in FROZEN mode.  diag, offd nullable.  gradE (nullable, [3n] as x|y|z planes) receives grad E
 * in UPDATE_LIMITER mode. */
int spray_fld_apply(spray_ctx* ctx, const double* m, const double* rho, const double* kappa, const double* E,
                    double c_light, spray_fld_kernel_mode_t kmode, spray_fld_limiter_mode_t lmode,
                    double* mu, double* y, double* diag, double* offd, double* gradE, void* stream);

/* (K9) parity exports, all device outputs, caller-allocated.
 * cell table: sorted_key[n], perm[n] (perm[i] = caller index of the particle in sorted slot i),
 *             cell_start[ncell], cell_end[ncell].  Any pointer may be NULL. */
int spray_get_cell_table(spray_ctx* ctx, uint32_t* sorted_key, uint32_t* perm, uint32_t* cell_start,
                         uint32_t* cell_end, void* stream);
/* count[a] = |N_sym(a)| (symmetric != 0) or |N_gather(a)| - 1 (symmetric == 0). */
int spray_neighbor_counts(spray_ctx* ctx, int symmetric, uint32_t* count, void* stream);
/* CSR neighbour lists: nbr[offsets[a] .. offsets[a]+count[a]) = caller ids of a's neighbours, ascending, self
 * excluded.  offsets = exclusive scan of the counts (u64[n]). */
int spray_neighbor_lists(spray_ctx* ctx, int symmetric, const uint64_t* offsets, uint32_t* nbr, void* stream);
/* Order-independent digest of each neighbour set (for full-size parity without moving the CSR lists):
 * dsum[a] = sum_b mix(id_b) mod 2^64, dxor[a] = xor_b mix(id_b), mix(v) = splitmix64(v): z = v + 0x9E3779B97F4A7C15,
 * z = (z ^ z>>30) * 0xBF58476D1CE4E5B9, z = (z ^ z>>27) * 0x94D049BB133111EB, z ^ z>>31;  id_b = caller index of b. */
int spray_neighbor_digest(spray_ctx* ctx, int symmetric, uint64_t* dsum, uint64_t* dxor, void* stream);

/* (N2) thermal-conduction sweep: the second term of eqs. (17)/(18), for one species,
 *       dudt_a = sum_b 4 m_b/(rho_a rho_b) * k_a k_b/(k_a + k_b) * (T_a - T_b) * x_ab . gradWbar(x_ab) / |x_ab|^2,
 *       gradWbar = (grad W(x_ab,h_a) + grad W(x_ab,h_b))/2,  over N_sym(a).
 * This is the Laplacian form eq. (16) with c = k, f = T, i.e. the FLD operator of spray_fld_apply (SYMMETRIC, FROZEN) with
 * mu = k and E = T, divided by rho_a; it is served by the same pair kernel.  Inputs m, rho, k (> 0), T in caller order;
 * dudt [out].  The electron-ion exchange term k^ei (T^e - T^i) of eqs. (17)/(18) is per-particle arithmetic left to the caller. */
int spray_conduction(spray_ctx* ctx, const double* m, const double* rho, const double* k, const double* T, double* dudt,
                     void* stream);

/* (N2, second half) implicit two-temperature heat transport: the backward-Euler system eqs. (28)-(29) as a
 * MATRIX-FREE operator (the paper assembles it for cuSPARSE ILU-BiCGSTAB; here it is applied, never stored), and its
 * right-hand side eqs. (33)-(34).  With C^s[g]_a = sum_b 4 m_b/(rho_a rho_b) k^s_a k^s_b/(k^s_a+k^s_b) (g_a - g_b) x_ab.gradWbar/|x_ab|^2
 * (the pair sum of spray_conduction over N_sym(a)), tau^s = dT^s/du^s and X_a = kei_a (g^e_a - g^i_a):
 *   which = SPRAY_COND_OPERATOR:  g^s = tau^s u^s,            out^i = u^i - dt (C^i[g^i] + X),  out^e = u^e - dt (C^e[g^e] - X)
 *        = Lambda^i u^i + sum_b chi^i_ab u^i_b - Gamma^e u^e  and  Lambda^e u^e + sum_b chi^e_ab u^e_b - Gamma^i u^i, eqs. (28)-(32)
 *        (eq. (29) prints + Gamma^i: DESIGN.md A37).  T_i, T_e are not read (may be NULL).
 *   which = SPRAY_COND_RHS:       g^s = T^s - tau^s u^s,      out^i = u^i + dt (C^i[g^i] + X) = b^i + c,  out^e = u^e + dt (C^e[g^e] - X) = b^e - c,
 *        eqs. (33)-(34), with (u, T) the state at time level N.
 * A Krylov or Jacobi solve of out_OPERATOR(u) = out_RHS is caller-side (two sweeps per application).
 * Inputs [n], caller order: m, rho, k_i, k_e (> 0), kei, dTdu_i, dTdu_e, T_i, T_e, u_i, u_e.  Outputs out_i, out_e [n], must not
 * alias inputs.  Errors: SPRAY_ERR_INVALID_ARG (NULL, unknown `which`, dt <= 0), SPRAY_ERR_ALLOC (scratch, first call). */
typedef enum { SPRAY_COND_OPERATOR = 0, SPRAY_COND_RHS = 1 } spray_cond_which_t;
int spray_conduction_implicit(spray_ctx* ctx, const double* m, const double* rho, const double* k_i, const double* k_e,
                              const double* kei, const double* dTdu_i, const double* dTdu_e, const double* T_i, const double* T_e,
                              const double* u_i, const double* u_e, double dt, spray_cond_which_t which, double* out_i, double* out_e,
                              void* stream);

/* (N3) continuity equation with the kernel-gradient-correction (KGC) filter, P:L207-L228:
 *       M_a = sum_b (m_b/rho_b) gradW(x_ab,h_a) (x) x_ba          eq. (40): row i = dW/dx_i, column j = (x_b - x_a)_j
 *       L_a = M_a^{-1}                                            eq. (40)
 *       drhodt_a = rho_a sum_b (m_b/rho_b) (v_a - v_b) . (L_a gradW(x_ab,h_a))      eq. (37) with eq. (39)
 * over N_gather(a) \ {a}, from the neighbour lists of the last spray_build_cells.  Since L_a does not depend on b the sum is
 * evaluated as L_a : sum_b (m_b/rho_b) (v_a - v_b) (x) gradW in the same sweep that accumulates M_a.  Where M_a is singular
 * (|det M_a| <= 1e-12; A28) the gradient is left uncorrected (L_a = I).
 * Inputs m, rho, vx, vy, vz in caller order.  drhodt [out, n]; L [out, nullable, 9 n]: L[(3 i + j) n + a] = (L_a)_ij;
 * drhodt_raw [out, nullable, n]: eq. (37) without the filter. */
int spray_kgc_continuity(spray_ctx* ctx, const double* m, const double* rho, const double* vx, const double* vy,
                         const double* vz, double* drhodt, double* L, double* drhodt_raw, void* stream);

/* (N1) implicit radiation step by Jacobi iteration, section 2.3 P:L268-L327.
 * Backward-Euler form of eqs. (47)-(48), i.e. eqs. (49)-(50), with the limiter frozen (mu[] given, A18).  Each of the
 * `niter` iterations (i) applies the FLD operator to the current iterate (spray_fld_apply FROZEN: Lambda_a, Gamma_a of eqs.
 * (51)-(52) over the neighbour lists of the last spray_build_cells), (ii) solves for every particle the quartic eq. (57)
 *       (1 - dt Lambda) a chi^4 + B chi - [E^n + dt Gamma + B T^n] = 0,   B = (1 - dt Lambda + dt rho c kappa_P) / (dt c kappa_P) / (dT/du)
 * for its positive root chi (eq. (56); the root "closest to u^n"; safeguarded Newton from the upper bound
 * min(C'^(1/4), C'/B'), because the closed form eqs. (58)-(60) cancels catastrophically for small roots -- DESIGN.md A25),
 * (iii) sets u = u^n + (chi - T^n)/(dT/du) (eq. (56)) and E = (u - u^n)/(dt c kappa_P) + a chi^4 (eq. (55)).
 * Inputs (caller order, length n): m, rho, mu (= c lambda/(rho kappa_R)), kappa_p, E_n, u_n, T_n, dTdu.
 * E [in/out]: the starting iterate (usually a copy of E_n) and, on return, E after niter iterations; u [out].
 * resid (nullable, DEVICE array of niter doubles): resid[k] = max_a |lhs - rhs| / |lhs| of eq. (49) for the iterate that
 * enters iteration k ("relative error of the difference between the two sides of equation (49)"), 0 for k = 0.
 * Requires dt, c_light, a_rad > 0, kappa_p > 0, dTdu > 0, niter >= 1.  E, u must not alias the inputs. */
int spray_rad_jacobi(spray_ctx* ctx, const double* m, const double* rho, const double* mu, const double* kappa_p,
                     const double* E_n, const double* u_n, const double* T_n, const double* dTdu, double dt, double c_light,
                     double a_rad, spray_fld_kernel_mode_t kmode, int niter, double* E, double* u, double* resid, void* stream);

/* (N4) mesh-free laser ray tracing and energy deposition, section 2.5.
 * f = n_e/n_c (dimensionless), kib = the inverse-bremsstrahlung absorption coefficient kappa^ib of eq. (70) per particle (an
 * input: nu^ei and the material data it needs are not in the paper).  Inputs m, rho, f, kib: [n], caller order.
 *   (1) gradient at the particles, as printed at P:L420:  G_a = sum_b (m_b/rho_b) f_b gradW(x_ab, h_a)  over N_gather(a)\{a}
 *       -> gradn (nullable, [3n] as x|y|z planes).
 *   (2) every ray q is a particle (x, v, P).  rays_in [7 nrays]: planes x, y, z, vx, vy, vz, P.  Per step of the fixed
 *       dt, with SPH interpolation at the ray's position over the particles with |x - x_a| < 2 h_a (own h, A30):
 *         G(x) = sum_a V_a G_a W(|x-x_a|,h_a);  kappa(x) = sum_a V_a kib_a W;  w_a = V_a W;  wsum = sum_a w_a
 *         v <- v - (c_light^2/2) G(x) dt              eq. (72)
 *         ds = |v| dt;  dE = P (1 - exp(-kappa(x) ds)) (eq. (71), A32);  P <- P - dE  (skipped when wsum = 0)
 *         edep_a += dE w_a / wsum                    ("based on the kernel weight", normalised: A33)
 *         x <- x + v dt with the new v (A31); periodic dimensions wrap
 *       A ray stops after nsteps steps, when P <= pmin, or once it has left [lo, hi) in a non-periodic dimension (A34).
 *   Outputs: edep [n] caller order (overwritten); rays_out [7 nrays] final state; steps_out (nullable, i64[nrays]) steps taken.
 * Uses the cell table of the last spray_build_cells (one warp per ray; rays are independent).  The deposit uses fp64
 * atomics: its summation order, hence its last bits, may differ from run to run; everything else is reproducible.
 * Errors: SPRAY_ERR_INVALID_ARG (NULL, nrays < 0, nsteps < 0, dt <= 0, c_light <= 0). nrays = 0 and n = 0 are valid. */
int spray_ray_deposit(spray_ctx* ctx, const double* m, const double* rho, const double* f, const double* kib, int64_t nrays,
                      const double* rays_in, double dt, int64_t nsteps, double c_light, double pmin, double* gradn, double* edep,
                      double* rays_out, int64_t* steps_out, void* stream);

/* Measurement aid: runs `iters` dependent DFMA per thread on `blocks` x `threads` threads
 * with 8 independent chains; out (device, [blocks*threads]) receives the sums so the work cannot be elided.
 * Used by bench.py to measure the sustained FP64 FMA peak the roofline is quoted against. */
int spray_fp64_peak_probe(int device, int blocks, int threads, int64_t iters, double* out, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* SPRAY_H_ */
