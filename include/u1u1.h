/*
 * u1u1.h -- C ABI of the B200-native U(1)xU(1) lattice field evolution library (libu1u1.so).
 *
 * The library evolves Saffin's dual-U(1) model (two complex scalars phi, psi with conjugate momenta
 * Pi, Psi; two gauge fields A, B stored as link phases theta = dx*A with electric fields E, H;
 * 20 fp32 words per site) on a periodic N^3 comoving lattice, as discretised in Correia & Martins,
 * arXiv:2208.01525 (cited below as PAPER.md:<line>), and computes the paper's in-loop diagnostics.
 * Every step of that path runs in hand-written sm_100a CUDA kernels; there is no CPU fallback.
 *
 * Conventions
 *   - Plain C types only.  Pointers are marked HOST or DEVICE.  The library never allocates or
 *     frees device memory: the caller owns `state_dev` and `scratch_dev` for the life of the context.
 *   - All work is enqueued on the CUDA stream given to u1u1_create (a cudaStream_t passed as void*;
 *     NULL = the legacy default stream).  Calls that fill HOST output synchronise that stream.
 *   - Every int-returning call returns 0 on success or a negative U1U1_E* code; no exception crosses
 *     the ABI.  u1u1_last_error(ctx) returns a human-readable message for the last failure.
 *   - Canonical state layout (export/import): float32 [20][N][N][N], x fastest, components
 *       0 phi_re 1 phi_im 2 Pi_re 3 Pi_im 4 psi_re 5 psi_im 6 Psi_re 7 Psi_im
 *       8..10 thetaA_xyz  11..13 E_xyz  14..16 thetaB_xyz  17..19 H_xyz
 *     theta_i = dx*A_i is NON-compact (never reduced mod 2 pi; the paper's gauge action is the
 *     non-compact one); E_i = dA_i/dtau.  The internal layout differs.
 *   - Time levels: positions (phi, psi, theta) at tau, momenta (Pi, Psi, E, H) at tau - dtau/2.
 */
#ifndef U1U1_H
#define U1U1_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define U1U1_OK 0
#define U1U1_EINVAL (-1)   /* bad argument, NULL pointer, struct_size mismatch                   */
#define U1U1_ESIZE (-2)    /* N unsupported, or a caller buffer is too small                     */
#define U1U1_EPARAM (-3)   /* couplings outside 0 <= kappa < sqrt(lambda1 lambda2)/2 */
#define U1U1_ESTATE (-4)   /* call out of order (e.g. step before init_fields / configure)        */
#define U1U1_ECUDA (-5)    /* a CUDA runtime call or kernel launch failed                         */
#define U1U1_EUNSTABLE (-6)/* dtau^2 (12/dx^2 + (lambda+2kappa) sigma^2 a^{2s}) >= 4: leapfrog unstable */

#define U1U1_DIAG_LEN 48   /* doubles written by u1u1_diagnostics  */
#define U1U1_GAUSS_LEN 8   /* doubles written by u1u1_gauss_violation */

typedef struct u1u1_ctx u1u1_ctx;

/* Model and run parameters.  Couplings are the a=1 values of PAPER.md:89 Eq. 12. */
typedef struct {
    uint32_t struct_size; /* = sizeof(u1u1_params); checked                                     */
    int32_t init_kind;    /* 0: |phi|=eta1,|psi|=eta2 with iid uniform phases
                             1: Gaussian-smoothed complex white noise normalised to the same moduli
                                (BASELINE.json config 3)                                         */
    double lambda1, lambda2; /* lambda_p0, lambda_q0   (Eq. 4)                       */
    double e1, e2;           /* e_p0, e_q0             (Eq. 2)                       */
    double eta1, eta2;       /* sigma_p, sigma_q: the symmetry-breaking scales     */
    double kappa;            /* kappa_0                (PAPER.md:52 Eq. 4, :89 Eq. 12)           */
    double dtau;             /* conformal timestep Delta eta                      */
    double tau_norm;         /* conformal time at which a = 1 (a = (tau/tau_norm)^p), > 0        */
    double friction;         /* every momentum is multiplied by this after the kick; 1 = off
                                (damping prephase of BASELINE.json configs 2 and 5)              */
    double smooth_width;     /* init_kind 1: Gaussian width in lattice units                     */
    int32_t smooth_trunc;    /* init_kind 1: kernel truncated at |d| <= smooth_trunc (<= 32)     */
    int32_t kernel_variant;  /* step kernel arithmetic (DESIGN.md sections 7-8), 0 .. 7:
                                0 = tiled, fp32 chain in DIFFERENCE FORM, SFU phasor (default: fp32 speed, Gauss
                                    residual within ~1-3x of the fp32 storage floor);
                                2 = tiled, plain fp32 chain, SFU phasor (Gauss residual ~30x the floor);
                                4 = tiled, fp64 kick chain, SFU phasor (Gauss residual AT the storage floor);
                                5 / 6 / 7 = 2 / 4 / 0 with libm sincosf instead of the SFU phasor;
                                1 / 3 = reference one-thread-per-site kernel in fp32 / fp64.
                                (The experimental switches that used to ride in the upper bits are no longer part of
                                this struct: include/u1u1_tuning.h.)                                  */
    int32_t range_reduce;    /* variant 0 only: explicit range reduction of the non-compact link phases in front of the
                                SFU sine / cosine -- phasor error 5e-7 at ANY |theta| instead of 6e-8 |theta| (identical
                                bits while |theta| < 2 pi, ~4 % slower).  0 = off (default), 1 = on,
                                2 = automatic: on from the first u1u1_diagnostics sweep that reports max |theta| > 10
                                (U1U1_D_MAX_THETA) until the next configure / init_fields.                */
    int32_t reserved;        /* 0 */
} u1u1_params;

/* Bytes of device memory the caller must provide for an N^3 lattice.
 * state  : 30 fp32 words/site (20 fields + a second copy of the 10 position words, ping-pong).
 * scratch: cell arrays (2 B/site) + a work area of 8 B/site -- winding codes for u1u1_export_windings, int32 segment
 *          labels and sizes for u1u1_pq_segments, two staging planes for the *_host copies -- plus the reduction
 *          partials. */
size_t u1u1_state_bytes(int32_t N);
size_t u1u1_scratch_bytes(int32_t N);

/* Optional second momentum buffer (10 fp32 words/site, DEVICE, 256-byte aligned; NULL detaches it).  With it,
 * u1u1_step advances TWO leapfrog steps per pass over the lattice (temporal blocking): a thread
 * block evaluates step 1 on its tile plus a one-site halo into shared memory and step 2 from there, so each site's 20
 * words make one HBM round trip per two steps (80 B per site-update instead of 160).  That kernel reads the halo
 * sites' momenta while neighbouring blocks update theirs, hence momenta go from one buffer to the other; the library
 * tracks which one is current.  Results are bit-identical to the one-step kernel's.  Cubic lattices, kernel_variant 0,
 * u1u1_step and u1u1_cool; an odd last step of a call takes the one-step kernel.  May be called before or after u1u1_configure; must hold
 * u1u1_aux_bytes(N).  1024^3: 43 GB on top of the 129 GB state (fits the 180 GB of a B200). */
size_t u1u1_aux_bytes(int32_t N);
int u1u1_set_aux(u1u1_ctx *ctx, void *aux_dev, size_t aux_bytes);

/* Create a context over caller-owned DEVICE buffers (256-byte aligned) and a CUDA stream.
 * Nothing is launched.  *ctx is a small HOST object, released by u1u1_destroy. */
int u1u1_create(u1u1_ctx **ctx, void *state_dev, size_t state_bytes, void *scratch_dev,
                size_t scratch_bytes, void *cuda_stream);
void u1u1_destroy(u1u1_ctx *ctx);
const char *u1u1_last_error(const u1u1_ctx *ctx); /* ctx may be NULL: returns the create() error */

/* Set lattice size, spacing and parameters without touching the fields (used before import_state).
 * N must be a multiple of 4 with 8 <= N <= 1024 and fit the buffers given to u1u1_create. */
int u1u1_configure(u1u1_ctx *ctx, int32_t N, double dx, const u1u1_params *params);

/* init_fields(seed, N, dx, params)  [north_star; PAPER.md:162]: configure, then generate the initial
 * condition on the device: scalars per params->init_kind from Philox4x32-10 keyed by `seed` with the
 * site's linear index (ix + N(iy + N iz)) as counter; Pi, Psi, theta, E, H = 0. */
int u1u1_init_fields(u1u1_ctx *ctx, uint64_t seed, int32_t N, double dx, const u1u1_params *params);

/* Replace parameters between phases (friction on/off, tau_norm, couplings); N, dx unchanged. */
int u1u1_set_params(u1u1_ctx *ctx, const u1u1_params *params);

/* Declare the conformal time and background of the CURRENT state without stepping: sets the scale
 * factor weights used by diagnostics / gauss_violation (c = cG = a(tau)^{2s}).  Needed only when a
 * state is imported and examined before any step. */
int u1u1_set_time(u1u1_ctx *ctx, double tau, double era_m, double s);

/* step(n, tau, era, s)  [north_star; Eq. 17-26]: n fused kick+drift leapfrog steps.
 * On entry positions are at `tau`, momenta at tau - dtau/2; step k uses tau_k = tau + k*dtau (fp64,
 * no accumulation).  era_m = m of a ∝ t^m (0 flat, 0.5 radiation, 2/3 matter, any 0 <= m < 1);
 * s = beta of PAPER.md:89 Eq. 12 (1 physical, 0 constant comoving width, < 0 core growth).
 * Asynchronous: returns after enqueueing. */
int u1u1_step(u1u1_ctx *ctx, int32_t n, double tau, double era_m, double s);

/* cool(n, dcool)  [PAPER.md:164-177 Eq. 27-30; reading R-20]: n explicit Euler steps of the diffusive
 * cooling that precedes the evolution in the paper's own initial-condition pipeline:
 *   dphi/deta = D-_j D+_j phi - lambda_p0/2 (|phi|^2 - sigma_p^2) phi,   dA_i/deta = -sum_j d-_j F_ij + 2 e_p0^2 Im(phi* D+_i phi)
 * and the mirror for (psi, B); no kappa term, no scale factor.  Runs in the fused step kernel with the kick
 * coefficients set to (0, 1) and the drift to dcool; on exit all momenta are zero.  The paper uses eta from -10
 * to 1 in steps of 1/30.  Needs dcool (12/dx^2 + max(lambda, 2 e^2) sigma^2) < 2 (explicit diffusion of the scalars
 * and of the links), else U1U1_EUNSTABLE.  Afterwards the diagnostic weights are those of a = 1 (no scale factor).
 * The high-expansion damping phase that follows is u1u1_step with era_m = 0.9 ... 0.95.
 * Asynchronous. */
int u1u1_cool(u1u1_ctx *ctx, int32_t n, double dcool);

/* diagnostics(out)  [north_star; PAPER.md:183-224 Eq. 31-37, :230-238]: out = HOST array of
 * U1U1_DIAG_LEN doubles, slots named by the U1U1_D_* enum below.  Uses the scale factor of the last
 * completed step (or of `tau_norm`-normalised a=1 before any step).  ONE read-only sweep over the state computes
 * everything, including the Gauss-law norms (slots U1U1_D_GAUSS..+7) and the pierced-cell arrays.  Synchronises
 * the stream. */
int u1u1_diagnostics(u1u1_ctx *ctx, double *out_host);

/* gauss_violation(out)  [north_star; PAPER.md:73-77 Eq. 9-10, :272]: out = HOST array of 8 doubles,
 * per sector (p then q): ||g||_2, ||rho||_2, max|g|, ||g||_2 / max(||rho||_2, ||div E||_2, tiny), with
 * g(x) = sum_i [E_i(x)-E_i(x-i)]/dx - rho(x), rho = 2 e0^2 cG Im(conj(phi) Pi) and
 * cG = c (1+delta)/(1+omega) of the last completed step.  Synchronises the stream. */
int u1u1_gauss_violation(u1u1_ctx *ctx, double *out_host);

/* gauss_violation_static: the same eight numbers (PAPER.md:73-77 Eq. 9-10, :272) for a caller that cannot allocate
 * device memory -- no context, no scratch buffer, and no cudaMalloc / cudaFree (or any allocating routine) inside.
 * Who that is: code living inside a host application whose own pool already holds all of HBM (a 1024^3 run with the
 * second momentum buffer leaves ~8 of 178 GiB), a monitor called from a loop that must not stall (cudaMalloc and
 * cudaFree synchronise the whole device), a tool that holds nothing but a checkpoint.  Such a caller cannot supply the
 * 10 B/site scratch buffer that u1u1_create wants, so this call reduces through a 256 KiB array built into the
 * library image instead (every GPU that loads libu1u1.so carries it until the process exits).
 *   state_canonical_dev  DEVICE, read only: float32 [20][N][N][N] in the canonical layout above (16-byte aligned)
 *   N                    multiple of 4, 8 <= N <= U1U1_STATIC_MAX_N; a larger N returns U1U1_ESIZE (the built-in array
 *                        holds 4 N partial rows and cannot grow)
 *   dx, e1, e2           lattice spacing and the a = 1 gauge couplings e_p0, e_q0, all > 0
 *   cG                   Gauss-law coefficient c (1+delta)/(1+omega) of the step that produced the state (what the
 *                        context tracks for u1u1_gauss_violation); a^{2s} for a state at rest, 1 in flat space
 *   out_dev              DEVICE, 8 doubles (8-byte aligned), layout as u1u1_gauss_violation; written by the last of the
 *                        two kernels this call enqueues on `cuda_stream`.  The call does NOT synchronise: read `out_dev`
 *                        after the stream has reached that point.
 *   err_host, err_len    optional HOST buffer that receives a message when the call fails (may be NULL / 0)
 * Returns 0 or a U1U1_E* code; nothing is enqueued on failure of the argument checks.
 * First call on a device: looks up the device address of the built-in array (cudaGetSymbolAddress, once per device,
 * with the current device).  Make that first call on each GPU during set-up, before any stream capture is begun.
 * Shared state: ALL calls in the process on the same GPU use the same array and find the previous call's partial
 * sums in it.  Every call overwrites the rows it reads, so nothing needs clearing and calls on ONE stream may follow
 * each other freely; two calls that can overlap on the GPU (different streams, different host threads without
 * ordering) race on the array and both results are garbage -- order them with an event. */
#define U1U1_STATIC_MAX_N 1024
int u1u1_gauss_violation_static(const void *state_canonical_dev, int32_t N, double dx, double e1, double e2, double cG,
                                double *out_dev, void *cuda_stream, char *err_host, size_t err_len);

/* Canonical-layout copies, DEVICE<->DEVICE (float32 [20][N][N][N]) and HOST<->DEVICE variants
 * (the host variants copy through the same stream and synchronise it). */
int u1u1_export_state(u1u1_ctx *ctx, void *dst_dev);
int u1u1_import_state(u1u1_ctx *ctx, const void *src_dev);
int u1u1_export_state_host(u1u1_ctx *ctx, void *dst_host);
int u1u1_import_state_host(u1u1_ctx *ctx, const void *src_host);

/* Fill the lattice with the periodic tiling of a smaller canonical state float32 [20][n_src][n_src][n_src] (DEVICE;
 * N must be a multiple of n_src): a relaxed small box as the initial condition of a large one, and -- because a tiled
 * state evolves as the tiling of the small evolution -- an exact full-size check of every kernel against a lattice
 * the oracle can afford. */
int u1u1_import_state_tiled(u1u1_ctx *ctx, const void *src_dev, int32_t n_src);

/* Canonical sub-block float32 [20][bz][by][bx] whose corner is site (x0,y0,z0), periodic wrap, to a
 * DEVICE buffer: lets a caller inspect a 1024^3 state (for which a full canonical copy does not fit
 * beside the state) -- used by the sampled full-size parity test. */
int u1u1_export_block(u1u1_ctx *ctx, int32_t x0, int32_t y0, int32_t z0, int32_t bx, int32_t by, int32_t bz,
                      void *dst_dev);

/* After u1u1_diagnostics (the per-plaquette codes are produced on the first request by a second sweep in export
 * mode): copy out the per-plaquette windings of `sector` (0 = p, 1 = q) as
 * int8 W[3][N][N][N] (orientation xy, yz, zx) and the near-branch-cut flags uint8 near[3][N][N][N]
 * (1 if any of the plaquette's four link angles lies within 1e-5 of +-pi), and the pierced-cell
 * array uint8 C[N][N][N].  DEVICE destinations; any of them may be NULL. */
int u1u1_export_windings(u1u1_ctx *ctx, int32_t sector, void *w_dev, void *near_dev, void *cells_dev);

/* pq_segments(min_cells, tolerant, out)  [PAPER.md:240-256, :390-394 "robust method"; reading R-21]:
 * after u1u1_diagnostics on the current state, label the connected regions (periodic 26-neighbourhood) of the
 * cells pierced by both string types -- exact overlap (tolerant = 0) or one cell of tolerance
 * (tolerant = 1, R-13b) -- and reduce them to out = HOST array of U1U1_SEG_LEN doubles:
 *   [0] N_pq     number of segments with at least min_cells cells          (Eq. 38)
 *   [1] L_pq     dx * sum over those segments of (N_cells - 1)             (off-by-one corrected)
 *   [2] l_pq     L_pq / N_pq (0 if there is none)                           (Eq. 38)
 *   [3] cells in those segments   [4] number of all segments   [5] number of all pq cells
 *   [6] cells of the largest segment
 *   [7] plain number of cells of the region mask (all regions): equals [5] for exact overlap; with tolerance it counts a
 *       one-cell-displaced pair twice, which is the reading R-21b replaced -- reported so both can be compared
 * The paper's production threshold is N_cells > 41 (min_cells = 42, L_pq > 20), Fig. 1 uses l_pq >= 3.5 (min_cells = 8).
 * A region's cell count is (its cells pierced by p + its cells pierced by q) / 2 (reading R-21b): the number of cells
 * for exact overlap, and the same length for a one-cell-displaced pair of lines as for a coincident pair.
 * Reuses the scratch work area (winding codes); the cell arrays stay valid.  Synchronises the stream. */
#define U1U1_SEG_LEN 8
int u1u1_pq_segments(u1u1_ctx *ctx, int32_t min_cells, int32_t tolerant, double *out_host);

/* After u1u1_pq_segments: int32 label[N][N][N] to a DEVICE buffer: -1 where the cell is not a pq cell, else the
 * linear index (x + N (y + N z)) of the smallest cell of its segment. */
int u1u1_export_labels(u1u1_ctx *ctx, void *labels_dev);

/* ---- z slabs: ONE lattice split over several GPUs.  Not the default: the
 * benchmark workload fits one GPU and runs there (north_star); this is the path to lattices that do not (PAPER.md:31:
 * 4096^3).  The global lattice is N x N x NZ_global, periodic; a rank's context owns nz_own consecutive z planes starting
 * at global plane z_first, stored with one halo plane below and above (buffer planes 0 .. nz_own + 1).  u1u1_step on a
 * slab advances the own planes by ONE step with the fused kernel and stores its top / bottom plane of the new positions
 * straight into the halo planes of the neighbouring slabs (plain stores through peer memory: NVLink when the neighbour
 * lives on another GPU), so there is no separate exchange pass.  Between two steps the caller must make sure that every
 * rank has finished the previous one (stream-ordered barrier / torch.distributed).  All slabs must have the same nz_own.
 * Available on a slab: set_params, step (n = 1, kernel_variant 0), init_slab, import_slab / export_slab, push_halos,
 * launch_count and the slab diagnostics below; the other diagnostics calls need a cubic lattice (U1U1_ESTATE). */
size_t u1u1_slab_state_bytes(int32_t N, int32_t nz_own);
int u1u1_configure_slab(u1u1_ctx *ctx, int32_t N, int32_t nz_own, int64_t z_first, double dx, const u1u1_params *params);
/* DEVICE pointers to the STATE buffers (as given to u1u1_create) of the slabs above and below (periodic: the top
 * slab's upper neighbour is the bottom slab; with a single slab both are its own buffer). */
int u1u1_set_slab_peers(u1u1_ctx *ctx, void *up_state_dev, void *dn_state_dev);
/* The random-phase initial condition of the GLOBAL lattice (same Philox counters = global site indices as
 * u1u1_init_fields) restricted to this slab's own planes; halo planes via u1u1_push_halos. */
int u1u1_init_slab(u1u1_ctx *ctx, uint64_t seed);
/* Canonical float32 [20][nz_own][N][N] (own planes only), DEVICE. */
int u1u1_export_slab(u1u1_ctx *ctx, void *dst_dev);
int u1u1_import_slab(u1u1_ctx *ctx, const void *src_dev);
/* Copy this slab's boundary planes of the current positions into the neighbours' halo planes (once, after init_slab /
 * import_slab on every rank; afterwards every step does it itself). */
int u1u1_push_halos(u1u1_ctx *ctx);

/* Diagnostics of a lattice in z slabs.  (1) every rank: u1u1_push_diag_halos (its top plane of E_z, H_z goes into the
 * momentum halo plane of the slab above: div E of the first own plane needs it), then a barrier; (2) every rank:
 * u1u1_slab_diagnostics_partial fills raw_host[U1U1_SLAB_NRAW] with the fused sweep's raw results over its own planes
 * (scratch must hold u1u1_slab_scratch_bytes); (3) the ranks reduce: SUM over the first U1U1_SLAB_NSUM values, MAX over
 * the rest; (4) u1u1_slab_diagnostics_finish turns the reduced array into the u1u1_diagnostics output for the lattice of
 * nz_global planes (the one-cell-tolerance counts, which would need cell-array halos, are NaN). */
#define U1U1_SLAB_NRAW 28
#define U1U1_SLAB_NSUM 24
size_t u1u1_slab_scratch_bytes(int32_t N, int32_t nz_own);
int u1u1_push_diag_halos(u1u1_ctx *ctx);
int u1u1_slab_diagnostics_partial(u1u1_ctx *ctx, double *raw_host);
int u1u1_slab_diagnostics_finish(u1u1_ctx *ctx, const double *raw_reduced_host, int64_t nz_global, double *out_host);

/* Number of kernel launches issued by this context so far (for bench.py's gpu_launches). */
uint64_t u1u1_launch_count(const u1u1_ctx *ctx);

/* Slots of the diagnostics array. */
enum {
    U1U1_D_TAU = 0,      /* conformal time of the positions                                      */
    U1U1_D_A,            /* scale factor a(tau)                                                  */
    U1U1_D_C,            /* c = a^{2s} used for the weights                                      */
    U1U1_D_SUMW_P,       /* sum over plaquettes |W^p|                             */
    U1U1_D_SUMW_Q,
    U1U1_D_CELLS_P,      /* cells pierced by p windings                                          */
    U1U1_D_CELLS_Q,
    U1U1_D_CELLS_PQ,     /* cells pierced by both (fast method, exact overlap)      */
    U1U1_D_NEAR_P,       /* plaquettes with a link angle within 1e-5 of the branch cut            */
    U1U1_D_NEAR_Q,
    U1U1_D_MAXW,         /* max |W| over both sectors (never >= 2 at equal tension) */
    U1U1_D_SUM_L,        /* sum_x L_x                         (Eq. 33)               */
    U1U1_D_SUM_KIN_L,    /* sum_x (|Pi|^2+|Psi|^2) L_x        (Eq. 37, W = L)        */
    U1U1_D_SUM_GRAD_L,   /* sum_x,i (|D+phi|^2+|D+psi|^2) L_x                                    */
    U1U1_D_SUM_KIN_V,    /* same with W = V_int = kappa0(|phi|^2-s_p^2)(|psi|^2-s_q^2) (:224)     */
    U1U1_D_SUM_GRAD_V,
    U1U1_D_SUM_VINT,
    U1U1_D_SUM_KIN,      /* energy components, no scale-factor weights, not multiplied by dx^3    */
    U1U1_D_SUM_GRAD,
    U1U1_D_SUM_ELEC,
    U1U1_D_SUM_MAG,
    U1U1_D_SUM_POT,
    U1U1_D_L_P,          /* derived, Eq. 31-37 ------------------------------- */
    U1U1_D_L_Q,
    U1U1_D_L_PQ,
    U1U1_D_XI_P,
    U1U1_D_XI_Q,
    U1U1_D_XI_PQ,
    U1U1_D_XI_W,
    U1U1_D_XI_L,
    U1U1_D_F_TOTAL,
    U1U1_D_F_P,
    U1U1_D_V2_L,
    U1U1_D_V2_PQ,
    U1U1_D_ENERGY,       /* dx^3 (kin+grad+elec+mag+pot): the flat-space Hamiltonian              */
    U1U1_D_CELLS_PQ_TOL_P, /* fast method with one cell of tolerance: pierced p cells  */
    U1U1_D_CELLS_PQ_TOL_Q, /* with a pierced q cell in their 3x3x3 neighbourhood; and q cells near p   */
    U1U1_D_L_PQ_TOL,     /* dx (tol_p + tol_q) / 2: equals L_pq for coincident AND for one-cell-displaced strings */
    U1U1_D_MAX_THETA,    /* largest |theta| of any link (non-compact phases drift in temporal gauge; the winding
                            sweep needs |theta| < 180 and u1u1_diagnostics fails with U1U1_ESTATE beyond)  */
    U1U1_D_GAUSS,        /* 8 slots: the u1u1_gauss_violation array of the same sweep (no second pass needed) */
    U1U1_D_V2_VALID = U1U1_D_GAUSS + 8, /* 1 * [V2_L usable] + 2 * [V2_PQ usable].  Eq. 36-37 is a velocity only
                            if the weight localises on strings: usable means R is finite with 0 <= R <= 1, i.e. 0 <= <v^2> <= 1.
                            When the weighted sums of |Pi|^2 and |D+ phi|^2 have opposite signs, or radiation dominates them
                            (e.g. config 5's early times, strings hundreds of lattice spacings wide), the bit is 0 and the
                            V2 slot -- still the raw 2R/(1+R) -- must not be read as a velocity.                        */
    U1U1_D_USED          /* number of slots in use (= U1U1_DIAG_LEN)                                */
};

#ifdef __cplusplus
}
#endif
#endif /* U1U1_H */
