/* include/mhd.h — C ABI of libmhd: the B200-native (sm_100a) hot path of the pseudo-spectral compressible
 * MHD solver of arXiv 1810.12707 ("G-MHD3D").
 *
 * What the library computes (citations: PAPER.md = the paper text; DESIGN.md = this repo's readings R1-R10):
 *   the right-hand side and explicit Adams-Bashforth step of the 3-D compressible, viscous, resistive MHD
 *   equations on a triply periodic N^3 box of side L (Sec. V Eq. 17-19; energy equation
 *   Eq. 12, in normalised units), discretised pseudo-spectrally: 3-D real FFTs, derivatives by
 *   multiplication with i*k, 2/3-rule dealiasing (L27; R5), real-space flux
 *   products, mu*lap(u) and eta*lap(B) diffusion, all in fp64 (Table I).
 *
 * Conventions
 *   - every field array is N^3 doubles laid out [z][y][x], x fastest, x_i = i*L/N (plan (Nz,Ny,Nx));
 *   - field order, conservative (kind 0): rho, mx, my, mz, E, Bx, By, Bz   with m = rho*u and
 *     E = P/(gamma-1) + rho|u|^2/2 + |B|^2/2 (1/8pi -> 1/2);
 *     primitive (kind 1): rho, ux, uy, uz, P, Bx, By, Bz;
 *   - `where` says what the caller's pointers are: MHD_HOST (0) = host memory (pageable or pinned),
 *     MHD_DEVICE (1) = device memory of the current CUDA device;
 *   - ownership: the caller owns every buffer it passes; the library copies in / out and never frees them.
 *     The context owns only small host metadata; all device storage lives inside the workspace handed to
 *     mhd_bind(), which the caller allocates (e.g. with torch) and must keep alive until mhd_destroy();
 *   - ordering: every call enqueues its work on the stream given to mhd_bind(); calls that return data to
 *     host memory (where = MHD_HOST, mhd_diagnostics) synchronise that stream before returning, calls with
 *     device pointers return as soon as the work is enqueued;
 *   - errors: every function returns MHD_OK (0) or a negative code and never throws, aborts or prints;
 *     mhd_last_error() returns a description of the last failure on that context;
 *   - threads: one context per host thread; contexts are independent.
 *   There is no CPU fallback: without a CUDA device every compute entry point returns MHD_ERR_CUDA.
 */
#ifndef MHD_H
#define MHD_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define MHD_OK 0
#define MHD_ERR_INVALID_ARG (-1)
#define MHD_ERR_NOT_BOUND (-2)
#define MHD_ERR_NO_FIELDS (-3)
#define MHD_ERR_CUDA (-4)
#define MHD_ERR_NOMEM (-5)

#define MHD_HOST 0
#define MHD_DEVICE 1

#define MHD_CONSERVATIVE 0
#define MHD_PRIMITIVE 1

/* workspace flags */
#define MHD_FLAG_DEFAULT 0u
/* The chunked ("out-of-core") pipeline, Sec. VII-C (L333-343, L375-379): the paper pages a working set larger
 * than device memory through CUDA unified memory; here storage is compact (only the modes inside the 2/3 mask), each
 * class of arrays is placed explicitly, and bricks / slabs of the host-resident classes are streamed through device
 * staging buffers on side streams.  Placement flags need MHD_FLAG_OUT_OF_CORE.           */
#define MHD_FLAG_OUT_OF_CORE 1u   /* chunked pipeline on compact storage; with no placement flag everything stays in HBM */
#define MHD_FLAG_STATE_ON_HOST 2u /* U^ and the Adams-Bashforth history live in pinned host memory                      */
#define MHD_FLAG_STAGE_STORAGE 8u /* chunked pipeline: also allocate the 8 compact accumulator arrays that the multi-stage
                                     integrators (MHD_OPT_INTEGRATOR = 1 RK4, 2 predictor-corrector) need beside U^ and the
                                     R^old arrays (which then hold the state at the start of the step): +50 % state storage  */
#define MHD_FLAG_WORK_ON_HOST 4u  /* the 16 work fields between the z and y passes live in pinned host memory           */
#define MHD_FLAG_RANKS(g) ((unsigned)((g) - 1) << 4) /* slab decomposition over g = 1..8 GPUs with PER-RANK storage: the context
                                     allocates only one rank's share (1/g of the state, 2/g of the work arrays: a brick-shaped
                                     and a slab-shaped set); needs MHD_FLAG_OUT_OF_CORE without host placement, and
                                     mhd_dist_config(rank, g) before any field call                                      */
#define MHD_FLAG_BUDGET_MIB(m) ((unsigned)(m) << 8) /* cap on the device workspace in MiB (0 = none): bounds the staging
                                     buffers; mhd_workspace_bytes() returns 0 if the placement cannot fit the budget     */

/* options for mhd_set_option() */
#define MHD_OPT_FUSED 1      /* 1 (default): fused kernels; 2: first-generation fused x sweep;
                                0: one kernel per step of the path (debug / bisect)                            */
#define MHD_OPT_PRUNE 2      /* 1 (default): skip pencils the 2/3 mask makes identically zero; 0: full sweeps  */
#define MHD_OPT_INTEGRATOR 3 /* 0 (default): Adams-Bashforth 2 with Euler start; 1: RK4; 2: predictor-corrector
                                (Table I; R6)                                 */

#define MHD_OPT_FUSE_CURRENT 4 /* 1 (default): J^ = M i k x B^ is built on load inside the inverse z pass (sweep S1);
                                0: separate kernel                                                            */

#define MHD_OPT_OOC_BRICK 5 /* chunked pipeline: largest number of ky columns per brick (0 = what the staging allows) */
#define MHD_OPT_OOC_SLAB 6  /* chunked pipeline: largest number of z planes per slab  (0 = what the staging allows) */

#define MHD_OPT_TRACER_SORT 11 /* re-sort the tracer storage by grid row every this many pushes (default 32; 0 = never):
                                  gather locality only, results do not depend on it (mhd_tracers_get returns id order) */

/* Equation-set variants of the paper (readings V1-V4).  Changing one resets the integrator history. */
#define MHD_OPT_EVOLVE 8  /* bit 0: Eq. 17-18 and the energy equation evolve, bit 1: Eq. 19 evolves (default 3).  2 = the
                             kinematic dynamo of PAPER.md L205 ("turn off Eq. 17 and 18"), 1 = hydrodynamic (L199)      */
#define MHD_OPT_STRESS 12 /* 1: the viscous terms of PAPER.md Eq. 11-12 (L92-96): + div(2 nu rho S) in the momentum equation and
                             the energy flux -2 nu rho u.S, with the traceless rate of strain S of Eq. 3-4 (L57-61) and nu = the
                             `mu` of mhd_init, instead of mu lap(u) (R3).  An unfused add-on pass (22 more transforms
                             per right-hand side); in-core contexts, Adams-Bashforth only                                  */
#define MHD_OPT_FORCE_K 9 /* integer mode number k_f >= 1 of the ABC forcing (default 1)                               */
/* parameters for mhd_set_param() */
#define MHD_PARAM_CS2 1       /* C_s^2 > 0: barotropic closure P = C_s^2 rho (Eq. 5, Eq. 18): E is carried
                                 but not evolved (R_E = 0); 0 (default): ideal gas, P from E (R1)             */
#define MHD_PARAM_FORCE_AMP 2 /* f0: external force rho f in the momentum equation (Eq. 18) with the ABC profile of
                                 L215, f = f0 (sin k z + cos k y, sin k x + cos k z, sin k y + cos k x), k = k_f 2 pi/L,
                                 and its work m.f in the energy equation; 0 (default): unforced.  In-core contexts only */

typedef struct mhd_ctx mhd_ctx; /* opaque, owned by the library */

/* Diagnostics record ("per grid" = volume means; L71 Eq. 9; R8). */
typedef struct {
    double t;          /* time = step * dt                                                     */
    long long step;    /* steps taken since the last mhd_set_fields                            */
    double ke;         /* <rho |u|^2 / 2>                                                      */
    double me;         /* <|B|^2 / 2>                                                          */
    double ie;         /* <P> / (gamma - 1)                                                    */
    double mass;       /* <rho>                                                                */
    double mom[3];     /* <m>                                                                  */
    double etot;       /* <E>                                                                  */
    double max_divb;   /* max over grid points of |d~x Bx + d~y By + d~z Bz| (dealiased spectral derivative) */
    double rho_min;    /* min rho                                                              */
    double p_min;      /* min P                                                                */
} mhd_diag;

/* Create a context.  N: power of two, 16 <= N <= 1024 (N = 8 is rejected: k_c = floor(8/3) = 2 leaves no usable band,
 * DESIGN.md section 1); L > 0; gamma > 1; mu, eta >= 0; dt > 0.
 * (mu, eta are the normalised 1/Re, 1/Rm of PAPER.md L140-152.)  Does not touch the GPU. */
int mhd_init(mhd_ctx **out, int N, double L, double gamma, double mu, double eta, double dt);

/* Device bytes the caller must provide to mhd_bind() for grid size N and the given flags. */
size_t mhd_workspace_bytes(int N, unsigned flags);
/* Page-locked host bytes mhd_bind() needs for the placement flags (0 if nothing lives on the host). */
size_t mhd_pinned_bytes(int N, unsigned flags);

/* Attach storage.  dev_workspace: device pointer, 256-byte aligned, >= mhd_workspace_bytes(N, flags);
 * cuda_stream: a cudaStream_t (NULL = legacy default stream); pinned_host/pinned_bytes: page-locked host
 * memory, 256-byte aligned, >= mhd_pinned_bytes(N, flags), for the host-resident classes of the chunked pipeline
 * (NULL/0 otherwise); the caller keeps it alive like the workspace.  Builds the twiddle tables (device work).
 * A context bound with MHD_FLAG_OUT_OF_CORE implements every call — including tracers, and the RK4 / predictor-corrector
 * integrators when MHD_FLAG_STAGE_STORAGE was given — except mhd_fft3d_*, the kinetic spectrum of mhd_diagnostics (needs an
 * unpruned transform) and the forcing / stress-tensor variants (refused with MHD_ERR_INVALID_ARG). */
int mhd_bind(mhd_ctx *ctx, void *dev_workspace, size_t bytes, void *cuda_stream, unsigned flags,
             void *pinned_host, size_t pinned_bytes);

int mhd_set_option(mhd_ctx *ctx, int option, int value);
int mhd_set_param(mhd_ctx *ctx, int param, double value);

/* Load a state.  f[i]: N^3 doubles each.  Primitive input is converted point-wise to conservative; each of the
 * 8 conservative fields is then dealias-projected, U <- IFFT(M FFT U) (R5).  Resets t = 0, step = 0
 * and the Adams-Bashforth history (the next step is a forward-Euler step, R6). */
int mhd_set_fields(mhd_ctx *ctx, int kind, int where, const double *const f[8]);

/* dU/dt of the current state in real space, 8 x N^3 doubles, conservative order.  Does not change the state,
 * the time or the integrator history. */
int mhd_rhs(mhd_ctx *ctx, int where, double *const out[8]);

/* Advance nsteps explicit steps of size dt.  mhd_step(a); mhd_step(b) is identical to mhd_step(a+b).
 * Only kernel launches; no host round trip. */
int mhd_step(mhd_ctx *ctx, int nsteps);

/* Current state in real space (kind as in mhd_set_fields). */
int mhd_get_fields(mhd_ctx *ctx, int kind, int where, double *const out[8]);

/* Diagnostics of the current state.  spec_kin / spec_mag (host pointers, may be NULL): shell spectra of
 * sqrt(rho)*u and of B, S(K) = sum over the full mode cube with floor(|n|+1/2) = K of 1/2 |w^(n)|^2 / N^6,
 * K = 0 .. nspec-1, nspec must equal mhd_nspec(N) = ceil(sqrt(3) N / 2) + 1; sum_K S(K) = ke resp. me. */
int mhd_diagnostics(mhd_ctx *ctx, mhd_diag *d, double *spec_kin, double *spec_mag, int nspec);
int mhd_nspec(int N);

/* ---- Diagnostics without a workspace -------------------------------------------------------------------------------
 * The scalar part of mhd_diagnostics (energies "per grid"; R8) for callers that can
 * give the library no device memory at all.  Everything above needs mhd_bind() and therefore a caller that can allocate
 * a workspace.  Some cannot: a monitoring or check-pointing hook that is only handed the eight field pointers of a solver
 * it does not own; a plug-in inside an application that reserved all of HBM for its own arena and exposes no allocator;
 * a health check that runs while another thread captures a CUDA graph, where cudaMalloc / cudaFree (which synchronise the
 * device) must not be called.  This one call needs no mhd_ctx and performs NO allocation of any kind (no cudaMalloc,
 * cudaFree, or library routine that allocates): the 80 KB of block partials that the two-stage reduction keeps between its
 * kernels live in a static __device__ array of libmhd.so, which every GPU that loads the library holds until the process
 * exits.
 *   n        grid points per field, 1 <= n <= MHD_NOALLOC_MAX_POINTS (2^30 = 1024^3, the library's largest grid); larger n is
 *            refused with MHD_ERR_INVALID_ARG and a message — the static array is fixed at 1024 blocks x 10 partials;
 *   gamma    adiabatic index > 1;
 *   dev_U    host array of 8 DEVICE pointers, conservative order (rho, mx, my, mz, E, Bx, By, Bz), n doubles each, read only;
 *   dev_out  DEVICE pointer to 10 doubles, written: ke, me, ie, mass, mom[0..2], etot (volume means as in mhd_diag),
 *            rho_min, p_min.  Bit for bit what mhd_diagnostics() reports for the same real-space arrays;
 *   cuda_stream  a cudaStream_t (NULL = legacy default stream); the two kernels are enqueued there and the call returns
 *            without synchronising; pointers belong to the current device;
 *   errbuf   optional host buffer (errbuf_len bytes) that receives a description when the return value is not MHD_OK.
 * Set-up: the FIRST call on each device looks up the device address of the static array (cudaGetSymbolAddress, with that
 * device current) and caches it; make that first call at start-up, before any stream capture begins.
 * Sharing: all calls on one GPU — from any thread, stream or context — use the same array.  It keeps the previous call's
 * partials; the first kernel overwrites every entry, so nothing needs clearing, but two calls whose kernels overlap on
 * the GPU (different streams, no ordering between them) race on it and return garbage.  Order them, e.g. by using one
 * stream. */
#define MHD_NOALLOC_MAX_POINTS (1LL << 30)
int mhd_energy_means_noalloc(long long n, double gamma, const double *const dev_U[8], double *dev_out,
                             void *cuda_stream, char *errbuf, size_t errbuf_len);

/* Stand-alone batched 3-D real FFT on DEVICE buffers (the FFT metric of BASELINE.json).
 *   r2c: real[i] (N^3 doubles) -> spec[i]: N*N*(N/2) complex doubles [kz][ky][kx], kx = 0..N/2-1, unnormalised
 *        forward transform F(n) = sum_x f(x) exp(-i k.x); the Nyquist column kx = N/2 goes to nyq[i]
 *        (N*N*8 complex, column 0 of each 8-wide row holds the value; may be NULL to drop it).
 *   c2r: the inverse with 1/N^3, Nyquist column taken as zero.  spec is destroyed (used as scratch).
 * prune != 0 restricts both to modes inside the 2/3 mask (others are not written / are read as zero). */
int mhd_fft3d_r2c(mhd_ctx *ctx, int nfields, const double *const real[], double *const spec[],
                  double *const nyq[], int prune);
int mhd_fft3d_c2r(mhd_ctx *ctx, int nfields, double *const spec[], double *const real[], int prune);

/* ---- Tracer particles (Sec. VI, readings T1-T4) ----------------
 * Passive particles with q = M = 1 that feel only the magnetic field of the grid (L241).  One push (L268-272) =
 *   1) corner index (i,j,k) = floor(x N/L) of the particle's unit cell;
 *   2) Eq. 20 (L251): cloud-in-cell interpolation of B from the 8 corner grids (weights = opposite sub-cell volumes /
 *      cell volume, corner indices wrapped periodically, L255);
 *   3) Eq. 21 (L259-265): t = B_p dt/2, s = 2t/(1+|t|^2), v_d = v + v x t, v(t+dt) = v + v_d x s;
 *   4) Eq. 22 (L266): x(t+dt) = x + v(t+dt) dt, wrapped into [0, L).
 * Storage: the caller provides mhd_tracers_bytes(np) device bytes (256-byte aligned; two sets of particle arrays, ids
 * and the scratch of the spatial sort, ~130 B per particle + 4 MB) and keeps them alive; pos / vel
 * arguments are 3 arrays (x, y, z components) of np doubles, host or device as `where` says.
 * mhd_tracers_set: positions are wrapped into [0, L); vel == NULL sets the initial velocity to the CIC interpolation
 *   of u = m/rho of the current state (L241; needs mhd_set_fields first).
 * While tracers are set, every step of mhd_step() first pushes them once with dt and the B of the state at the START
 * of that step (t_n), then advances the fields.  mhd_tracers_push() pushes nsteps times in the B of the current state
 * without advancing the fields (one kernel; the gather benchmark).
 * Chunked (MHD_FLAG_OUT_OF_CORE) contexts: the buffer of mhd_tracers_bind must be mhd_tracers_bytes(np) +
 * mhd_tracers_field_bytes(ctx) long — the tracers then keep their own real-space copies of B (and of rho, m for the
 * initial velocity), filled slab by slab at the start of every step; not available on a decomposed context. */
size_t mhd_tracers_bytes(long long np);
size_t mhd_tracers_field_bytes(const mhd_ctx *ctx);   /* 0 for in-core contexts */
int mhd_tracers_bind(mhd_ctx *ctx, long long np, void *dev_buffer, size_t bytes);   /* np = 0 detaches */
int mhd_tracers_set(mhd_ctx *ctx, int where, const double *const pos[3], const double *const vel[3]);
int mhd_tracers_get(mhd_ctx *ctx, int where, double *const pos[3], double *const vel[3]);
int mhd_tracers_push(mhd_ctx *ctx, int nsteps);

/* ---- Slab decomposition over several GPUs (not in the paper) -----------------
 * One process per GPU.  A context bound with MHD_FLAG_OUT_OF_CORE (everything in device memory) becomes rank `rank` of
 * `world`: it owns a contiguous share of the compact ky axis for the z passes, the assembly and the update (phases A, C)
 * and a contiguous share of the z planes for the y passes and the fused x sweep (phase B).  Between the phases the work
 * arrays are transposed across ranks by an all-to-all that THE CALLER performs (torch.distributed over NCCL) on device
 * buffers packed / unpacked by the library.  One step:
 *     [phase A]  pack(0,11) -> all-to-all -> unpack(0,11)  phase B  pack(1,16) -> all-to-all -> unpack(1,16)  phase C(next)
 * phase C with arg != 0 also runs phase A of the next step on the updated bricks (then the next step starts at pack).
 * mhd_set_fields (every rank passes the full fields; only its z planes are read) must be followed by the exchange
 * (1, 8) and MHD_DIST_PHASE_STORE; mhd_get_fields (only the rank's z planes of `out` are written) must be preceded by
 * MHD_DIST_PHASE_STATE_Z and the exchange (0, 8).  mhd_step / mhd_rhs / mhd_diagnostics return MHD_ERR_INVALID_ARG on
 * a decomposed context.  Counts are in doubles, per peer, in rank order (the split sizes of the all-to-all). */
#define MHD_DIST_PHASE_A 0        /* U^ -> J^ on load, inverse z pass of own ky bricks -> work[0..10]              */
#define MHD_DIST_PHASE_B 1        /* inverse y, fused x sweep, forward y on own z planes -> work[0..15]             */
#define MHD_DIST_PHASE_C 2        /* forward z, assembly, explicit update of own bricks (+ next phase A if arg != 0) */
#define MHD_DIST_PHASE_STORE 3    /* mhd_set_fields, second half: forward z + projection into the compact state    */
#define MHD_DIST_PHASE_STATE_Z 4  /* mhd_get_fields, first half: inverse z pass of the state -> work[0..7]          */
int mhd_dist_config(mhd_ctx *ctx, int rank, int world);
int mhd_dist_phase(mhd_ctx *ctx, int phase, int arg);
int mhd_dist_counts(mhd_ctx *ctx, int dir, int nfields, long long *send_counts, long long *recv_counts);
int mhd_dist_pack(mhd_ctx *ctx, int dir, int nfields, double *dev_sendbuf);
int mhd_dist_unpack(mhd_ctx *ctx, int dir, int nfields, const double *dev_recvbuf);
int mhd_dist_ranges(mhd_ctx *ctx, int rank, int *ky_lo, int *ky_hi, int *z_lo, int *z_hi);   /* shares of any rank */
/* Direct exchange (at most 8 ranks): delta_bytes[s] = address of rank s's workspace MINUS this rank's, as mapped into THIS
 * process (CUDA IPC / peer access over NVLink; all ranks bind workspaces of the same size).  Phases A, B, C then store every
 * output row straight into the work arrays of the rank that owns it (P2P stores from inside the z-pass and forward-y
 * kernels, overlapping the transform tile by tile): the step needs no pack, collective or unpack, only a barrier where an
 * exchange would be (after A, after B): [A] barrier B barrier C(next).  NULL switches back to the packed exchange.
 * mhd_set_fields / mhd_get_fields keep using the packed exchange. */
int mhd_dist_peers(mhd_ctx *ctx, const long long *delta_bytes);
/* Lets kernels of the current device dereference memory of `peer_device` (cudaDeviceEnablePeerAccess; "already enabled"
 * is not an error).  Needed once per peer GPU before the direct exchange; a no-op for the current device itself. */
int mhd_dist_enable_peer_access(mhd_ctx *ctx, int peer_device);

/* Bytes the chunked pipeline has copied host->device / device->host so far (0 for an in-core context). */
int mhd_transfer_bytes(const mhd_ctx *ctx, long long *h2d, long long *d2h);

/* Number of kernels this context has launched so far (for the bench's gpu_launches claim). */
long long mhd_launch_count(const mhd_ctx *ctx);
const char *mhd_last_error(const mhd_ctx *ctx);
int mhd_destroy(mhd_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* MHD_H */
