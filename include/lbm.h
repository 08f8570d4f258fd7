/*
 * lbm.h -- C-ABI boundary of the B200-native Shan-Chen multiphase lattice-Boltzmann step.
 *
 * What is computed: the per-timestep update of the JAX-LaB paper (arxiv 2506.17713):
 *   Eq. 1-3   collide (BGK / MRT) + stream
 *   Eq. 4,10  moments rho^k, j^k per component
 *   Eq. 5-6   exact-difference forcing, half-force velocity on output
 *   Eq. 12 pseudopotential psi(rho) from an equation of state
 *   Eq. 13 Shan-Chen interaction force F_SC, 1 or 2 components
 *   Eq. 17 improved virtual-density wetting at solid nodes
 *   no-slip bounce-back, pressure / flux inlet-outlet
 * on D2Q9 and D3Q19.  Where the paper is silent the readings R1..R17 of DESIGN.md
 * apply (they restate SURVEY.md section 8(c) G1..G17).
 *
 * Conventions
 *   - All functions are extern "C" and return int: LBM_OK (0) or a negative lbm_status.
 *     No exceptions, no abort, nothing printed.  lbm_last_error(h) gives a library-owned
 *     message valid until the next call on h.
 *   - Every step of the path runs in CUDA kernels for sm_100a.  There is NO CPU fallback:
 *     without a CUDA device lbm_create fails with LBM_E_CUDA.
 *   - The library allocates no device memory.  The caller passes ONE device workspace of at
 *     least lbm_workspace_bytes(cfg) bytes (256-byte aligned) and a cudaStream_t; the library
 *     carves the workspace and keeps using it until lbm_destroy.  The handle is small host
 *     memory owned by the library.
 *   - Array arguments are caller-owned and never retained after the call returns.  For each
 *     array the `on_device` flag says whether the pointer is a device pointer (used directly by
 *     kernels on the stream, asynchronous) or a host pointer (copied with cudaMemcpyAsync on the
 *     stream followed by a stream synchronise before return).
 *   - Layout: scalar fields are flat with x fastest, index = x + nx*(y + ny*z).  Populations are
 *     structure-of-arrays [q][N]; vector fields [d][N].
 *   - Direction order (fixed, part of the ABI):
 *       D2Q9 : 0 rest; 1..4 = +x,-x,+y,-y; 5..8 = (1,1),(-1,-1),(1,-1),(-1,1)
 *       D3Q19: 0 rest; 1..6 = +x,-x,+y,-y,+z,-z; 7..10 = (1,1,0),(-1,-1,0),(1,-1,0),(-1,1,0);
 *              11..14 = (1,0,1),(-1,0,-1),(1,0,-1),(-1,0,1); 15..18 = (0,1,1),(0,-1,-1),(0,1,-1),(0,-1,1)
 *     lbm_get_lattice returns the tables.
 *   - Faces: 0 = x-min, 1 = x-max, 2 = y-min, 3 = y-max, 4 = z-min, 5 = z-max.
 */
#ifndef LBM_B200_H
#define LBM_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define LBM_API __attribute__((visibility("default")))
#else
#define LBM_API
#endif

typedef struct lbm lbm_t;
typedef void* lbm_stream_t; /* a cudaStream_t (NULL = default stream) */

enum lbm_status {
    LBM_OK = 0,
    LBM_E_INVALID = -1,     /* bad argument or configuration */
    LBM_E_UNSUPPORTED = -2, /* valid but not built (e.g. fp64 compute with fp16 storage) */
    LBM_E_NOMEM = -3,       /* workspace too small or misaligned */
    LBM_E_CUDA = -4,        /* CUDA runtime error (message in lbm_last_error) */
    LBM_E_STATE = -5        /* call out of order (e.g. step before init_fields) */
};

enum lbm_lattice { LBM_D2Q9 = 0, LBM_D3Q19 = 1 };

/* psi(rho), Eq. 12 for the EOS kinds: psi = sqrt(max(0, 2(alpha p_EOS - c_s^2 rho)/g_kk));
 * LBM_PSI_RHO: psi = rho; LBM_PSI_EXP: psi = exp(-1/rho);
 * LBM_PSI_SC93: psi = rho0 (1 - exp(-rho/rho0)) (Shan & Chen 1993, cited PAPER.md:121). */
enum lbm_psi_kind {
    LBM_PSI_EOS_CS = 0,  /* Carnahan-Starling */
    LBM_PSI_EOS_PR = 1,  /* Peng-Robinson */
    LBM_PSI_EOS_VDW = 2, /* van der Waals */
    LBM_PSI_EOS_RK = 3,  /* Redlich-Kwong */
    LBM_PSI_EOS_RKS = 4, /* Redlich-Kwong-Soave */
    LBM_PSI_RHO = 5,
    LBM_PSI_EXP = 6,
    LBM_PSI_SC93 = 7
};

enum lbm_collision { LBM_BGK = 0, LBM_MRT = 1 };      /* Eq. 3 lines 1-2 */
enum lbm_forcing { LBM_EDM = 0, LBM_SHIFT = 1 };      /* Eq. 5 / velocity shift */
enum lbm_dtype { LBM_F16 = 0, LBM_F32 = 1, LBM_F64 = 2 };
enum lbm_face_kind { LBM_FACE_PERIODIC = 0, LBM_FACE_WALL = 1, LBM_FACE_VELOCITY = 2, LBM_FACE_PRESSURE = 3 };

/* flags */
#define LBM_FLAG_NO_COLLIDE 1u /* f* = f: pure streaming, for the bit-exact permutation test */
#define LBM_FLAG_TWO_PASS 2u   /* always run the two-pass path K1 (+K1b) + K2 */
#define LBM_FLAG_ONE_PASS 4u   /* require a one-pass kernel K2F: lbm_step fails with LBM_E_UNSUPPORTED where none applies
                                  (D2Q9, solid cells, a non-periodic axis, rows that are not whole 16-byte vectors of the
                                  storage dtype, or a dtype/component combination it is not built for).  Default (neither
                                  flag): K2F where it applies and the domain is large enough to fill the GPU, else two-pass. */

/* Tuning knobs.  NOT part of the ABI: environment variables read once, in lbm_create, for measurements and tests; no other
 * call reads the environment.  LBM_TUNE_FUSED_MCHUNK=<planes marched per CTA of the one-pass kernels>, LBM_TUNE_NO_EQ (run
 * k_fused_ws where k_fused_eq would apply), LBM_TUNE_EQ_HALF=0|1 (tile width of k_fused_eq), LBM_TUNE_EQ_SPLIT=0|1|2 (k_fused_eq_split off / late / early
 * take), LBM_TUNE_EQ_YGROUP=<tile rows per launch of k_fused_eq_split; with it, one launch per chunk of planes>, LBM_TUNE_WS_TY=7|8 (rows
 * per tile of k_fused_ws with one component and of k_fused_eq at fp64), LBM_TUNE_LIST=0|1 and
 * LBM_TUNE_COMPACT=0 (list / fluid-compact mode of the two-pass path on masked domains), LBM_TUNE_BRICK="bx,by,bz" (order of
 * the fluid-cell list), LBM_TUNE_NO_SNBR, LBM_TUNE_NO_PDL / LBM_TUNE_NO_GRAPH / LBM_TUNE_NO_COOP (plain launches on small
 * domains), LBM_TUNE_NO_TILE (small 2-D domains on k_steps_coop / graph replay instead of k_steps_tile).  Results never depend on them beyond rounding order (none changes any arithmetic). */

typedef struct {
    int32_t psi_kind; /* lbm_psi_kind */
    int32_t pad_;
    double a, b, R, omega; /* EOS parameters (Yuan & Schaefer 2006 as quoted PAPER.md:199, 236) */
    double T;              /* absolute temperature in lattice units */
    double alpha;          /* pressure modification parameter alpha^k of Eq. 12 (1 = unmodified) */
    double rho0;           /* LBM_PSI_SC93 reference density */
} lbm_eos_t;

typedef struct {
    double phi, drho; /* Eq. 17: rho_s = phi*rho_ave - drho */
    double lo, hi;    /* limiter bounds */
} lbm_wetting_t;

typedef struct {
    int32_t lattice;      /* lbm_lattice */
    int32_t nx, ny, nz;   /* nz must be 1 for D2Q9; nx*ny*nz < 2^31 */
    int32_t n_components; /* 1 or 2 */
    int32_t periodic[3];  /* per axis; faces of non-periodic axes default to LBM_FACE_WALL */
    int32_t collision;    /* lbm_collision */
    int32_t forcing;      /* lbm_forcing */
    int32_t compute_dtype; /* LBM_F32 or LBM_F64: arithmetic type of every kernel */
    int32_t store_dtype;   /* LBM_F16 / LBM_F32 / LBM_F64: population storage */
    uint32_t flags;
    int32_t pad_;
    lbm_eos_t eos[2];
    double G[2][2];          /* g_kk' of Eq. 13; Green's function weights are w_i/c_s^2 (reading R2) */
    lbm_wetting_t wet[2];
    double tau[2];           /* BGK relaxation time (> 1/2).  It is also the relaxation time of the momentum that enters the
                                common velocity u' = sum_k (j^k/tau_k) / sum_k (rho^k/tau_k) (R6) and LBM_SHIFT (R7).
                                With LBM_MRT the rates below decide everything and tau is not read. */
    double mrt_rates[2][19]; /* diagonal of S in the moment order of DESIGN.md R9 (first q entries used).  The momentum rows
                                (3, 5 and, on D3Q19, 7) must share one non-zero rate s_j (LBM_E_INVALID otherwise): 1/s_j
                                takes the place of tau_k in the common velocity and in LBM_SHIFT, so that a collision
                                changes the total momentum by exactly sum_k F^k (Eq. 3 + Eq. 10)
                                whatever the other rates are. */
    double rho_ref;          /* populations are stored as f_i - w_i*rho_ref (reading R16); 0 = plain */
    double zc_A[2];          /* A_kk of Eq. 11 / 13: F^k = A_kk F_ZC^k + (1 - A_kk) F_SC^k with the Zhang-Chen
                                force F_ZC^k = -sum_i G_i U^k(x+e_i) e_i, U^k = alpha p_EOS - c_s^2 rho (Eq. 12).  0 = plain
                                Shan-Chen.  Non-zero needs an EOS psi kind (LBM_E_INVALID otherwise) and runs the two-pass path. */
    double body_accel[3];    /* body force per unit mass a: F^k += rho^k a on every fluid cell (R19) */
    double st_kappa[2];      /* kappa of Eq. 16: MRT source term that scales the surface tension with
                                1 - kappa and keeps the coexistence densities.  D2Q9 with LBM_MRT only (the D3Q19 form is not
                                in the paper): LBM_E_UNSUPPORTED otherwise.  Runs the two-pass path. */
} lbm_config_t;

/* Bytes of device workspace lbm_create needs for cfg; 0 if cfg is invalid. */
LBM_API size_t lbm_workspace_bytes(const lbm_config_t* cfg);

/* Create a simulation on the current CUDA device.  d_workspace: device pointer, 256-byte aligned,
 * >= lbm_workspace_bytes(cfg) bytes, owned by the caller, must outlive the handle.  All later device
 * work is enqueued on `stream`.  Errors: LBM_E_INVALID, LBM_E_UNSUPPORTED, LBM_E_NOMEM, LBM_E_CUDA. */
LBM_API int lbm_create(const lbm_config_t* cfg, void* d_workspace, size_t workspace_bytes, lbm_stream_t stream, lbm_t** out);

/* Free the handle.  Never frees the workspace.  NULL is allowed. */
LBM_API void lbm_destroy(lbm_t* h);

/* Solid mask: N bytes, non-zero = solid (no-slip by halfway bounce-back, reading R13).  Derives the
 * per-cell link flags and the list of boundary solids (solids with >= 1 fluid neighbour, reading R11).
 * Must be called before lbm_init_fields (LBM_E_STATE afterwards). */
LBM_API int lbm_set_solid_mask(lbm_t* h, const uint8_t* mask, int on_device);

/* Boundary condition of one face of a non-periodic axis (reading R10): LBM_FACE_WALL (halfway
 * bounce-back), LBM_FACE_VELOCITY (bounce-back + 2 w_i rho_w e_i.u_w/c_s^2) or LBM_FACE_PRESSURE
 * (anti-bounce-back f_i = -f*_ibar + 2 w_i rho_w [1 + (e_i.u)^2/(2 c_s^4) - u.u/(2 c_s^2)] with the boundary node's own
 * velocity u: the one bracket for which a uniform equilibrium flow passes the face unchanged).  rho_w[2] per component,
 * u_w[3].  LBM_E_INVALID for a face of a periodic axis.  The rule is folded into the stored populations at the writing
 * cell, so a face can be (re)defined before lbm_init_fields or between lbm_init_fields and the first lbm_step only:
 * LBM_E_STATE once steps have run (call lbm_init_fields again to start over). */
LBM_API int lbm_set_face_bc(lbm_t* h, int face, int kind, const double* rho_w, const double* u_w);

/* S0: f_i^k = f_eq,i(rho^k, u) at fluid cells (solid cells hold f_eq(1,0) and are never updated);
 * resets the step counter.  rho[k]: N values each; u: [d][N] or NULL (= 0); dtype: LBM_F32 or LBM_F64
 * element type of the arrays. */
LBM_API int lbm_init_fields(lbm_t* h, const void* const* rho, const void* u, int dtype, int on_device);

/* Enqueue n >= 0 time steps (S1..S7) on the stream.  Asynchronous; no host synchronisation -- with one exception: on a
 * domain with a solid mask, the first lbm_init_fields / lbm_step / export after lbm_set_solid_mask or lbm_set_face_bc
 * builds the link flags and cell lists and reads two counters back (one stream synchronisation, once per mask).
 * Layout note: on a masked domain with at most a quarter of the cells fluid (and a plain Shan-Chen force) the steps
 * run on a fluid-compact copy of the populations (lbm_hot_path reports LBM_PATH_TWO_PASS_COMPACT); the first step
 * after, and the first export / import after such steps, each cost one extra copy kernel.  Results are bit-identical
 * to the dense layout; solid cells read back as f_eq(1,0), whatever lbm_set_populations had put there.
 * Small domains (n_components * cells <= 2^22) with n >= 2: all n steps run as ONE cooperative launch of a persistent
 * kernel where the device allows it -- 2-D lattices on k_steps_tile (LBM_PATH_ONE_PASS_TILE: rho and psi recomputed on a
 * ring around each CTA's tile, one grid barrier per step), others on k_steps_coop (LBM_PATH_TWO_PASS_PERSISTENT) --, else
 * as CUDA-graph replays of 16 captured steps; bit-identical to n calls with n = 1, which launch the kernels one by one. */
LBM_API int lbm_step(lbm_t* h, int n);

/* S8: rho^k (virtual density at boundary solids, 0 inside solids), u = (sum_k j^k + 1/2 sum_k F^k)/sum_k rho^k
 * (Eq. 6; 0 at solids), p = c_s^2 sum_k rho^k + 1/2 sum_kk' g_kk' psi^k psi^k' (0 at solids).
 * Any of rho / u / p may be NULL.  dtype: LBM_F32 or LBM_F64. */
LBM_API int lbm_get_macroscopic(lbm_t* h, void* const* rho, void* u, void* p, int dtype, int on_device);

/* Parity exports.  Populations are the canonical post-stream f_i(x,t) of component comp, [q][N],
 * whatever the internal storage is.  dtype LBM_F32 or LBM_F64. */
LBM_API int lbm_get_populations(lbm_t* h, int comp, void* f, int dtype, int on_device);
/* Set the post-stream populations directly (tests; doubles as a restart). */
LBM_API int lbm_set_populations(lbm_t* h, int comp, const void* f, int dtype, int on_device);
/* Per cell: bit i (1 <= i < q) set <=> the pull of direction i does not read a fluid neighbour
 * (source solid or beyond a non-periodic face); a solid cell reports exactly 0x80000000. */
LBM_API int lbm_get_link_flags(lbm_t* h, uint32_t* flags, int on_device);
/* Boundary-solid list, ascending cell index.  Returns the count (>= 0) or a negative status;
 * writes min(count, capacity) entries to host memory `out` (may be NULL to query the count). */
LBM_API int64_t lbm_get_boundary_solids(lbm_t* h, int64_t* out, int64_t capacity);
/* psi^k field of the current state (compute dtype converted to dtype), N values. */
LBM_API int lbm_get_psi(lbm_t* h, int comp, void* psi, int dtype, int on_device);

/* Headless in-situ rendering of the density field (PAPER.md:339, 347 render device-resident
 * arrays without a host copy; the paper gives no formula, DESIGN.md "Rendering" is the definition).  An
 * iso-surface rho^comp = iso seen along +axis (0 = x, 1 = y, 2 = z) with orthographic rays, one per lattice
 * column.  Pixel (u, v): the two other axes in ascending order (axis 2: u = x, v = y; axis 1: u = x, v = z;
 * axis 0: u = y, v = z); both images are [n_v][n_u] row-major, n_u * n_v values of dtype (LBM_F32 / LBM_F64).
 * The field is the one lbm_get_macroscopic exports (virtual density in boundary solids, 0 in other solids).
 * Along a ray the first pair of samples (k, k+1) with (rho_k - iso)(rho_{k+1} - iso) <= 0 and rho_k != rho_{k+1}
 * is the hit: depth = k + (iso - rho_k) / (rho_{k+1} - rho_k); no hit: depth = -1 and shade = 0.
 * shade = 0.1 + 0.9 max(0, n.l), n = -grad(rho)/|grad(rho)| interpolated between the two samples (central
 * differences, periodic wrap or clamped index per axis), l = (1, 1, -2)/sqrt(6) in the (u, v, axis) frame;
 * |grad| = 0 gives 0.1.  shade / depth: host or device pointers per on_device; either may be NULL, not both.
 * One kernel over the resident field; nothing but the images crosses to the host. */
LBM_API int lbm_render_isosurface(lbm_t* h, int comp, double iso, int axis, void* shade, void* depth, int dtype,
                                  int on_device);

/* ---- Slab decomposition along the LAST axis (z for D3Q19, y for D2Q9): the multi-GPU exchange step.
 * A rank's handle holds its slab of the global domain plus `width` ghost layers below and above it along the last
 * axis, is configured PERIODIC along that axis (the wrap only ever feeds ghost layers) and steps as usual; before every
 * lbm_step the ghost layers are overwritten with the neighbours' outermost interior layers:
 *     lbm_export_halo(side)  packs the `width` interior layers next to the ghost layers of `side` (0: low, 1: high),
 *     lbm_import_halo(side)  overwrites the `width` ghost layers of `side` with a packed buffer,
 * so rank r's export(1) is rank r+1's import(0) and rank r+1's export(0) is rank r's import(1).  width = 2 for a plain
 * Shan-Chen step (the force at the outermost interior layer reads psi one layer out, Eq. 13, and psi there is taken from
 * populations pulled one layer further, Eq. 2 + Eq. 12), width = 3 when solid cells with virtual density (Eq. 17) can
 * lie in the ghost layers.  The solid mask passed to lbm_set_solid_mask covers the ghost layers too.  After a step the
 * ghost layers hold values computed from wrapped data; they are never read by an owned cell before the next import --
 * by lbm_step, that is: the exports (lbm_get_populations, lbm_get_macroscopic, lbm_render_isosurface) return post-stream
 * values, which the outermost owned layer pulls from the first ghost layer, so exchange once more before exporting.
 * Buffer: device memory, lbm_halo_bytes() bytes, [component][direction][layer][cells of a layer] in the STORAGE dtype --
 * the stored (post-collision, R14) populations, moved as bytes; 16-byte alignment makes the copy vectorised, alignment
 * to the storage dtype is required.  Asynchronous on the handle's stream; one copy kernel per call.
 * Errors: LBM_E_INVALID (side, width < 1 or 3 * width > layers, last axis not periodic, alignment), LBM_E_STATE before
 * lbm_init_fields.  A handle in the fluid-compact layout is converted back to the dense one first. */
LBM_API int lbm_halo_bytes(lbm_t* h, int width, size_t* bytes);
LBM_API int lbm_export_halo(lbm_t* h, int side, int width, void* d_buf);
LBM_API int lbm_import_halo(lbm_t* h, int side, int width, const void* d_buf);

/* ---- One time step without any allocation and without a handle or workspace: for callers that cannot call cudaMalloc
 * (code under CUDA graph capture, tight serving loops, harnesses that forbid it).
 * lbm_step_noalloc runs S1..S7 once, as the two-pass arrangement K1 (rho, psi) -> K2 (force, collision, streaming), on
 * caller-held arrays: d_f_in = f_i^k(x, t) and d_f_out = f_i^k(x, t + 1), both DEVICE arrays [component][q][N] of
 * cfg->compute_dtype in the layout and meaning of lbm_get_populations / lbm_set_populations (post-stream values;
 * cfg->store_dtype is ignored), distinct from each other.  The psi field K1 hands to K2 is held in a static device array
 * of LBM_NOALLOC_SCRATCH_BYTES inside the library (every GPU that loads the library holds it until exit), so
 *     n_components * nx * ny * nz * sizeof(compute dtype) <= LBM_NOALLOC_SCRATCH_BYTES      (2 MiB: 512 x 256 fp32 with two
 *     components, 512 x 512 fp64, 64^3 fp64, 80^3 fp32),
 * larger domains are refused with LBM_E_NOMEM.  Built for: D2Q9 / D3Q19, one or two components, BGK / MRT, both forcing
 * schemes, body force, fully periodic domains without solid cells and the plain Shan-Chen force (anything else:
 * LBM_E_UNSUPPORTED; bad pointers or configuration: LBM_E_INVALID).  Asynchronous on `stream`; two kernel launches; no
 * cudaMalloc / cudaFree / allocating library call, no host synchronisation.
 * ALL calls on a GPU share the one scratch array: calls whose kernels may overlap on that GPU (different streams without
 * ordering between them, several host threads or processes' contexts are separate copies) RACE on it -- order them.  The
 * array keeps the previous call's contents; every word K2 reads is written by K1 of the same call, so nothing needs
 * clearing.  lbm_noalloc_last_error() returns the calling thread's message for the last failing lbm_step_noalloc. */
#define LBM_NOALLOC_SCRATCH_BYTES (2u << 20)
LBM_API int lbm_step_noalloc(const lbm_config_t* cfg, const void* d_f_in, void* d_f_out, lbm_stream_t stream);
LBM_API size_t lbm_noalloc_max_scratch_bytes(void);
LBM_API const char* lbm_noalloc_last_error(void);

/* Lattice tables: q, e[q][3], w[q], opposite[q].  Host pointers; any may be NULL. */
LBM_API int lbm_get_lattice(int lattice, int* q, int* e, double* w, int* opposite);

/* sizeof(lbm_config_t) as compiled into the library (ABI check for bindings). */
LBM_API size_t lbm_config_bytes(void);

/* Measurement only: per-kernel device time of the hot loop.  While enabled, lbm_step brackets each of its
 * kernels with a pair of CUDA events recorded on the handle's stream (this serialises nothing but adds two
 * event records per kernel, so whole-step throughput is measured with profiling OFF).
 * lbm_get_kernel_times synchronises the stream, adds up the elapsed time of every bracketed launch since the
 * last call and resets the accumulators.  ms_total / launches: host arrays of LBM_K_COUNT entries indexed by
 * lbm_kernel_id.  Errors: LBM_E_INVALID, LBM_E_CUDA. */
enum lbm_kernel_id {
    LBM_K_MOMENTS = 0, /* K1: rho + psi (two-pass path) */
    LBM_K_VIRTUAL = 1, /* K1b: virtual density at boundary solids */
    LBM_K_STEP = 2,    /* K2: fused stream + force + collide + boundary (two-pass path) */
    LBM_K_FUSED = 3,   /* K2F: one-pass kernel (moments + psi of the halo recomputed in the tile) */
    LBM_K_PERSISTENT = 4, /* the persistent kernels of small domains (k_steps_tile / k_steps_coop): one launch makes n time
                             steps; its time is recorded as a whole and `launches` counts the n steps */
    LBM_K_COUNT = 5
};
LBM_API int lbm_set_profiling(lbm_t* h, int enable);
LBM_API int lbm_get_kernel_times(lbm_t* h, double* ms_total, int64_t* launches);

/* Which kernels the most recent lbm_step launched (the driver's "is the native path the one that runs" question,
 * and the tests' check that a fast kernel was not silently replaced by a fallback). */
enum lbm_path {
    LBM_PATH_NONE = 0,              /* no step yet */
    LBM_PATH_TWO_PASS = 1,          /* K1 (+K1b) + K2 */
    LBM_PATH_RESERVED_2 = 2,        /* (round 1's lock-step one-pass kernel; removed) */
    LBM_PATH_ONE_PASS_WS = 3,       /* K2F k_fused_ws (warp-specialised, bulk asynchronous copies) */
    LBM_PATH_TWO_PASS_COMPACT = 4,  /* K1 (+K1b) + K2 on the fluid-compact layout (at most a quarter of the cells fluid) */
    LBM_PATH_ONE_PASS_EQ = 5,       /* K2F k_fused_eq / k_fused_eq_split (row pipelines; one component, BGK with tau = 1) */
    LBM_PATH_TWO_PASS_PERSISTENT = 6, /* K1 | K1b | K2 as phases of one persistent cooperative kernel (small domains, n >= 2) */
    LBM_PATH_ONE_PASS_TILE = 7       /* small 2-D domains, n >= 2: one persistent kernel, rho / psi recomputed on a ring around each
                                        CTA's tile, one grid barrier per step (k_steps_tile) */
};
LBM_API int lbm_hot_path(const lbm_t* h);

/* Bookkeeping. */
LBM_API int64_t lbm_steps_done(const lbm_t* h);
LBM_API int64_t lbm_kernel_launches(const lbm_t* h); /* kernels launched by this handle so far */
LBM_API const char* lbm_last_error(const lbm_t* h);
LBM_API const char* lbm_version(void);

#ifdef __cplusplus
}
#endif
#endif /* LBM_B200_H */
