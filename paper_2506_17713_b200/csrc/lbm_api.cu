// lbm_api.cu -- the C-ABI of include/lbm.h: configuration checks, workspace carving, boundary
// preprocessing kernels, and the launch sequence of the hot loop (K1 -> K1b -> K2 per step).
// No device memory is allocated here; everything lives in the caller's workspace.
#include "../../include/lbm.h"
#include "lbm_launch.cuh"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <queue>
#include <new>
#include <string>
#include <vector>

using namespace lbmk;

namespace {

constexpr size_t ALIGN = 256;
constexpr int CHUNK_CELLS = 1 << 21;  // staging granularity for host / converted transfers

size_t align_up(size_t v) { return (v + ALIGN - 1) / ALIGN * ALIGN; }
size_t dtype_bytes(int dt) { return dt == LBM_F16 ? 2 : dt == LBM_F32 ? 4 : 8; }

struct Carve {
    size_t f[2], psi, rho, flags, bsolid, flist, nbr, snbr, mask, counter, stage_a, stage_b, total;
};

}  // namespace

// Tuning knobs: environment variables read ONCE, in lbm_create (include/lbm.h lists them; not part of the ABI)
struct Tune {
    int mchunk = 0;        // LBM_TUNE_FUSED_MCHUNK: planes marched per CTA of the one-pass kernels (0 = cost model)
    int list = -1;         // LBM_TUNE_LIST: force list mode on (1) / off (0)
    int compact = -1;      // LBM_TUNE_COMPACT=0: keep the dense layout where compact mode would apply
    int eq = -1;           // LBM_TUNE_NO_EQ=1 -> 0: k_fused_ws where k_fused_eq would apply
    int eq_half = -1;      // LBM_TUNE_EQ_HALF: force full-width (0) / half-width (1) tiles of k_fused_eq
    int ws_ty = -1;        // LBM_TUNE_WS_TY: rows per tile of k_fused_ws (fshape.ty or one fewer; -1: chosen per domain)
    int eq_ygroup = -1;    // LBM_TUNE_EQ_YGROUP: k_fused_eq_split launched per chunk of planes and per group of this many tile rows (0: one launch)
    int eq_split = -1;     // LBM_TUNE_EQ_SPLIT: k_fused_eq_split off (0) / on with late (1) / early (2) take; -1: chosen per domain
    bool no_snbr = false;  // LBM_TUNE_NO_SNBR: K1b of the compact mode on the dense rho field
    bool no_pdl = false;   // LBM_TUNE_NO_PDL / LBM_TUNE_NO_GRAPH / LBM_TUNE_NO_COOP: plain launches on small domains
    bool no_graph = false;
    bool no_coop = false;
    bool no_tile = false;  // LBM_TUNE_NO_TILE: small 2-D domains on k_steps_coop / graph replay instead of k_steps_tile
    int brick[3] = {32, 16, 16};   // LBM_TUNE_BRICK="bx,by,bz": bricks of the fluid list's order (bx = 0: ascending cell index)
    static Tune from_env() {
        Tune t;
        auto geti = [](const char* name, int dflt) { const char* e = std::getenv(name); return e ? std::atoi(e) : dflt; };
        t.mchunk = geti("LBM_TUNE_FUSED_MCHUNK", 0);
        t.list = geti("LBM_TUNE_LIST", -1);
        t.compact = geti("LBM_TUNE_COMPACT", -1);
        t.eq = std::getenv("LBM_TUNE_NO_EQ") ? 0 : -1;
        t.eq_half = geti("LBM_TUNE_EQ_HALF", -1);
        t.eq_split = geti("LBM_TUNE_EQ_SPLIT", -1);
        t.eq_ygroup = geti("LBM_TUNE_EQ_YGROUP", -1);
        t.ws_ty = geti("LBM_TUNE_WS_TY", -1);
        t.no_snbr = std::getenv("LBM_TUNE_NO_SNBR") != nullptr;
        t.no_pdl = std::getenv("LBM_TUNE_NO_PDL") != nullptr;
        t.no_graph = std::getenv("LBM_TUNE_NO_GRAPH") != nullptr;
        t.no_coop = std::getenv("LBM_TUNE_NO_COOP") != nullptr;
        t.no_tile = std::getenv("LBM_TUNE_NO_TILE") != nullptr;
        if (const char* e = std::getenv("LBM_TUNE_BRICK")) {
            int v[3] = {0, 1, 1};
            if (std::sscanf(e, "%d,%d,%d", &v[0], &v[1], &v[2]) >= 1) { t.brick[0] = v[0]; t.brick[1] = std::max(1, v[1]); t.brick[2] = std::max(1, v[2]); }
        }
        return t;
    }
};

struct lbm {
    lbm_config_t cfg;
    Tune tune;
    int q, d, N;
    long long plane;
    size_t sbytes, cbytes;
    cudaStream_t stream;
    char* ws;
    Carve cv;
    int cur;
    int vec;   // cells per thread in the hot kernels (1 or the dtype's vector width)
    FusedShape fshape;   // tile of the one-pass kernel K2F (vec = 0: not built for this configuration)
    int fmchunk;         // planes marched per CTA
    bool use_fused;      // decided in prepare()
    bool eq_half;        // k_fused_eq with half-width tiles and two CTAs per SM
    int eq_ygroup;       // k_fused_eq_split: tile rows per launch (0: the whole domain in one launch)
    int ws_ty;           // k_fused_ws: rows per tile chosen by plan_fused (0: fshape.ty)
    int eq_split;        // 0: k_fused_eq; 1 / 2: k_fused_eq_split (front / back warps per row) with late / early take
    bool feq;            // one component, BGK, tau = 1: the collision result is f_eq(rho, u' + du) (k_fused_eq applies)
    int last_path;       // lbm_hot_path: what the last lbm_step ran
    // launch-bound (small) domains: GRAPH_STEPS time steps captured once into a CUDA graph and replayed
    cudaGraphExec_t gexec;
    int gcur;            // buffer parity the graph was captured at
    int64_t glaunches;   // kernels per replay
    bool gvalid, gfailed;
    bool tile_failed;    // k_steps_tile does not apply (3-D, more tiles than resident CTAs, no cooperative launch)
    bool coop_failed;    // the cooperative launch of the persistent small-domain kernel is not available
    bool initialized, has_solid, bnd, dirty, force_rho;
    int nbsolid;
    int nfluid;       // fluid cells (masked domains)
    bool use_list;    // hot kernels iterate over the fluid-cell list (porous domains)
    bool pdl;         // lbm_step on a small domain: hot kernels are launched as programmatic dependents
    bool has_bmask;   // fluid-neighbour masks of the boundary solids are stored behind their list
    bool compact_on;  // lbm_step keeps the populations in fluid-list order (lbm_compact.cuh)
    bool is_compact;  // layout of the current population buffer
    long long nbr_stride;
    long long snbr_stride;   // 0: K1b of the compact mode gathers the dense rho field
    int face_kind[6];
    double face_rho[6][2], face_u[6][3];
    int64_t steps, launches;
    std::string err;
    // kernel parameter block, rebuilt only when the configuration-derived part changes (params_valid = false)
    bool params_valid;
    KParams<float> pf32;
    KParams<double> pf64;
    // measurement only (lbm_set_profiling): event pairs around hot-loop kernels
    bool profiling;
    std::vector<cudaEvent_t> ev_pool;
    struct EvPair { int kid; int n; cudaEvent_t a, b; };   // n: time steps the bracketed launch made
    std::vector<EvPair> ev_pending;
    double k_ms[LBM_K_COUNT];
    int64_t k_cnt[LBM_K_COUNT];
};

// Halo layers of the slab decomposition (lbm_export_halo / lbm_import_halo): `rows` chunks of `row_units` units of U bytes,
// chunk r at src + r * src_pitch -> dst + r * dst_pitch (pitches in units).  Pure data movement in the storage dtype.
template <class U>
__global__ void __launch_bounds__(256) k_halo_copy(U* __restrict__ dst, const U* __restrict__ src, long long rows, long long row_units,
                                                   long long src_pitch, long long dst_pitch) {
    const long long total = rows * row_units;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const long long r = t / row_units, c = t - r * row_units;
        dst[r * dst_pitch + c] = src[r * src_pitch + c];
    }
}

namespace {

int q_of(int lattice) { return lattice == LBM_D2Q9 ? 9 : 19; }

int check_config(const lbm_config_t* c) {
    if (!c) return LBM_E_INVALID;
    if (c->lattice != LBM_D2Q9 && c->lattice != LBM_D3Q19) return LBM_E_INVALID;
    if (c->nx < 1 || c->ny < 1 || c->nz < 1) return LBM_E_INVALID;
    if (c->lattice == LBM_D2Q9 && c->nz != 1) return LBM_E_INVALID;
    if ((long long)c->nx * c->ny * c->nz >= (1LL << 31) - 64) return LBM_E_INVALID;
    if (c->n_components < 1 || c->n_components > 2) return LBM_E_INVALID;
    if (c->collision != LBM_BGK && c->collision != LBM_MRT) return LBM_E_INVALID;
    if (c->forcing != LBM_EDM && c->forcing != LBM_SHIFT) return LBM_E_INVALID;
    if (c->compute_dtype != LBM_F32 && c->compute_dtype != LBM_F64) return LBM_E_INVALID;
    if (c->store_dtype != LBM_F16 && c->store_dtype != LBM_F32 && c->store_dtype != LBM_F64) return LBM_E_INVALID;
    if (c->compute_dtype == LBM_F32 && c->store_dtype == LBM_F64) return LBM_E_INVALID;
    if (c->compute_dtype == LBM_F64 && c->store_dtype == LBM_F16) return LBM_E_UNSUPPORTED;
    for (int k = 0; k < c->n_components; ++k) {
        const lbm_eos_t& e = c->eos[k];
        if (e.psi_kind < LBM_PSI_EOS_CS || e.psi_kind > LBM_PSI_SC93) return LBM_E_INVALID;
        if (e.psi_kind <= LBM_PSI_EOS_RKS) {
            if (!(c->G[k][k] < 0.0)) return LBM_E_INVALID;  // R4: g_kk < 0 under the root
            if (!(e.b > 0.0) || !(e.R > 0.0) || !(e.T > 0.0)) return LBM_E_INVALID;
        }
        if (e.psi_kind == LBM_PSI_SC93 && !(e.rho0 > 0.0)) return LBM_E_INVALID;
        if (c->zc_A[k] != 0.0 && e.psi_kind > LBM_PSI_EOS_RKS) return LBM_E_INVALID;   // U of Eq. 12 needs an EOS
        if (c->st_kappa[k] != 0.0 && (c->lattice != LBM_D2Q9 || c->collision != LBM_MRT)) return LBM_E_UNSUPPORTED;
        if (!(c->tau[k] > 0.5)) return LBM_E_INVALID;
        if (c->collision == LBM_MRT) {   // the momentum rows share one non-zero rate (lbm.h: mrt_rates)
            const int nj = c->lattice == LBM_D2Q9 ? 2 : 3;
            if (!(c->mrt_rates[k][3] > 0.0)) return LBM_E_INVALID;
            for (int a = 1; a < nj; ++a)
                if (c->mrt_rates[k][3 + 2 * a] != c->mrt_rates[k][3]) return LBM_E_INVALID;
        }
    }
    return LBM_OK;
}

// Bricks of the fluid-cell list's visit order (VisitOrder in the preprocessing kernels): 32 x 16 x 16 cells by default
// (measured on config 4, K2: ascending cell order 1.45 ms, 16x4x4 1.40, 8x8x8 1.34, 16x8x8 1.29, 32x16x16 1.22, 32^3 1.20);
// every dimension is at most BRICK_MAX, which is what the workspace is sized for.
constexpr int BRICK_MAX = 64;
long long brick_volume(const lbm_config_t& c, const int (&b)[3]) {   // positions the brick order visits (brick-padded domain)
    if (b[0] <= 0) return (long long)c.nx * c.ny * c.nz;
    auto up = [](long long n, int m) { return (n + m - 1) / m * m; };
    return up(c.nx, b[0]) * up(c.ny, b[1]) * up(c.nz, c.nz > 1 ? b[2] : 1);
}

Carve carve(const lbm_config_t& c) {
    Carve v{};
    const size_t N = (size_t)c.nx * c.ny * c.nz;
    const size_t q = q_of(c.lattice), nc = c.n_components;
    const size_t plane = (N + 63) / 64 * 64;
    const size_t sb = dtype_bytes(c.store_dtype), cb = dtype_bytes(c.compute_dtype);
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off += align_up(bytes); return o; };
    v.f[0] = take(nc * q * plane * sb);
    v.f[1] = take(nc * q * plane * sb);
    v.psi = take(nc * N * cb);
    v.rho = take(nc * N * cb);
    v.flags = take(N * 4);
    v.bsolid = take(N * 4);
    const int bmax[3] = {BRICK_MAX, BRICK_MAX, BRICK_MAX};
    const size_t npos = (size_t)std::max<long long>((long long)N, brick_volume(c, bmax));
    v.flist = take(N * 4 + ((npos + 1023) / 1024 + 1) * 4);   // fluid-cell list + per-block counts of its compaction
    v.nbr = take((q - 1) * (N / 4 + 64) * 4);   // neighbour table of the compact mode (fluid fraction <= 1/4)
    v.snbr = take((q - 1) * (N / 4 + 64) * 4);  // ... and of its boundary solids (used when there are at most N/4 of them)
    v.mask = take(N);
    v.counter = take(256);
    const size_t chunk = std::min<size_t>(N, CHUNK_CELLS);
    v.stage_a = take(q * chunk * 8);
    v.stage_b = take(q * chunk * 8);
    v.total = off;
    return v;
}

double eos_tc(int kind, double a, double b, double R) {
    switch (kind) {
        case LBM_PSI_EOS_CS: return 0.3773 * a / (b * R);
        case LBM_PSI_EOS_PR: return 0.0778 / 0.45724 * a / (b * R);
        case LBM_PSI_EOS_VDW: return 8.0 / 27.0 * a / (b * R);
        case LBM_PSI_EOS_RK: return std::cbrt(std::pow(0.08664 / 0.42748 * a / (b * R), 2.0));
        case LBM_PSI_EOS_RKS: return 0.08664 / 0.42748 * a / (b * R);
    }
    return 1.0;
}

template <class L>
void lattice_weights(double* w) {
    for (int i = 0; i < L::Q; ++i) w[i] = (double)L::WN[i] / (double)L::WD;
}

// M^-1 S M = sum_r (s_r / |M_r|^2) M_r^T M_r split by the parity of the moment polynomial of row r (R9):
// even rows act on (f_0, f_a + f_b) only, odd rows on (f_a - f_b) only (a = 2p+1, b = 2p+2).
//   ce[P][Q] = sum_{r even} c_r M_r,i(P) M_r,i(Q),  i(0) = 0, i(P) = 2P-1;   co[P][Q] = sum_{r odd} c_r M_r,2P+1 M_r,2Q+1
template <class L>
void mrt_blocks(const double* rates, double (&ce)[10][10], double (&co)[9][9]) {
    constexpr int NP = (L::Q - 1) / 2;
    for (auto& row : ce) for (double& v : row) v = 0.0;
    for (auto& row : co) for (double& v : row) v = 0.0;
    for (int r = 0; r < L::Q; ++r) {
        double m[19], n2 = 0.0;
        for (int i = 0; i < L::Q; ++i) { m[i] = 0.5 * mrt_entry2<L>(r, i); n2 += m[i] * m[i]; }
        bool even = true;
        for (int pq = 0; pq < NP; ++pq)
            if (m[2 * pq + 1] != m[2 * pq + 2]) even = false;
        const double cr = rates[r] / n2;
        if (even) {
            for (int P = 0; P <= NP; ++P)
                for (int Q = 0; Q <= NP; ++Q) ce[P][Q] += cr * m[P ? 2 * P - 1 : 0] * m[Q ? 2 * Q - 1 : 0];
        } else {
            for (int P = 0; P < NP; ++P)
                for (int Q = 0; Q < NP; ++Q) co[P][Q] += cr * m[2 * P + 1] * m[2 * Q + 1];
        }
    }
}

template <class CT>
KParams<CT> make_params(const lbm* h, int in_buf, int out_buf) {
    KParams<CT> p;
    std::memset(&p, 0, sizeof p);
    const lbm_config_t& c = h->cfg;
    p.nx = c.nx; p.ny = c.ny; p.nz = c.nz; p.N = h->N;
    for (int a = 0; a < 3; ++a) p.periodic[a] = c.periodic[a] ? 1 : 0;
    p.plane = h->plane;
    p.f_in = h->ws + h->cv.f[in_buf];
    p.f_out = h->ws + h->cv.f[out_buf];
    p.psi = reinterpret_cast<CT*>(h->ws + h->cv.psi);
    p.rho = reinterpret_cast<CT*>(h->ws + h->cv.rho);
    p.flags = reinterpret_cast<const uint32_t*>(h->ws + h->cv.flags);
    p.bsolid = reinterpret_cast<const int*>(h->ws + h->cv.bsolid);
    p.nbsolid = h->nbsolid;
    p.flist = reinterpret_cast<const int*>(h->ws + h->cv.flist);
    p.nfluid = h->nfluid;
    p.nbr = reinterpret_cast<const uint32_t*>(h->ws + h->cv.nbr);
    p.nbr_stride = h->nbr_stride;
    p.cplane = h->nbr_stride;
    p.compact = 0;
    p.forcing = c.forcing == LBM_SHIFT ? 1 : 0;
    p.write_rho = (h->nbsolid > 0 || h->force_rho) ? 1 : 0;
    double w[19];
    if (c.lattice == LBM_D2Q9) lattice_weights<D2Q9>(w);
    else lattice_weights<D3Q19>(w);
    for (int i = 0; i < h->q; ++i) p.wref[i] = (CT)(w[i] * c.rho_ref);
    for (int k = 0; k < c.n_components; ++k) {
        // relaxation time of the momentum (common velocity R6, velocity shift R7): tau for BGK, 1 / (rate of the
        // momentum rows) for MRT -- only then does a collision change the total momentum by exactly sum_k F^k
        const double tmom = c.collision == LBM_MRT ? 1.0 / c.mrt_rates[k][3] : c.tau[k];
        p.tau[k] = (CT)tmom;
        p.inv_tau[k] = (CT)(1.0 / tmom);
        for (int kp = 0; kp < c.n_components; ++kp) p.G[k][kp] = (CT)c.G[k][kp];
        // BGK as one linear combination (lbm_hot.cuh collide): EDM  f* = (1-w) f + (w-1) feq(u') + feq(u'+du),
        // SHIFT  f* = (1-w) f + w feq(u' + tau du), w = 1/tau
        const double om = 1.0 / c.tau[k];
        p.c_keep[k] = (CT)(1.0 - om);
        p.c_feq_a[k] = (CT)(c.forcing == LBM_SHIFT ? om : om - 1.0);
        p.c_feq_b[k] = (CT)(c.forcing == LBM_SHIFT ? 0.0 : 1.0);
        if (c.collision == LBM_MRT) {
            double ce[10][10], co[9][9];
            if (c.lattice == LBM_D2Q9) mrt_blocks<D2Q9>(c.mrt_rates[k], ce, co);
            else mrt_blocks<D3Q19>(c.mrt_rates[k], ce, co);
            for (int r = 0; r < 10; ++r)
                for (int q2 = 0; q2 < 10; ++q2) p.mrt_ce[k][r][q2] = (CT)ce[r][q2];
            for (int r = 0; r < 9; ++r)
                for (int q2 = 0; q2 < 9; ++q2) p.mrt_co[k][r][q2] = (CT)co[r][q2];
            if (c.lattice == LBM_D3Q19)
                for (int r = 0; r < 19; ++r) {
                    const double n2 = (double)mrt_norm2<D3Q19>(r);
                    p.mrt_c1[k][r] = (CT)((1.0 - c.mrt_rates[k][r]) / n2);
                    p.mrt_c2[k][r] = (CT)(c.mrt_rates[k][r] / n2);
                    p.mrt_c3[r] = (CT)(1.0 / n2);
                }
        }
        const lbm_eos_t& e = c.eos[k];
        p.psi_kind[k] = e.psi_kind;
        p.eos_a[k] = (CT)e.a;
        p.eos_b[k] = (CT)e.b;
        p.eos_RT[k] = (CT)(e.R * e.T);
        p.eos_sqrtT[k] = (CT)std::sqrt(e.T > 0 ? e.T : 1.0);
        p.eos_alpha[k] = (CT)e.alpha;
        p.eos_rho0[k] = (CT)e.rho0;
        p.eos_inv_gkk2[k] = c.G[k][k] != 0.0 ? (CT)(2.0 / c.G[k][k]) : (CT)0;
        double aalpha = e.a;
        if (e.psi_kind == LBM_PSI_EOS_PR || e.psi_kind == LBM_PSI_EOS_RKS) {
            const double tc = eos_tc(e.psi_kind, e.a, e.b, e.R);
            const double m = e.psi_kind == LBM_PSI_EOS_PR
                                 ? 0.37464 + 1.54226 * e.omega - 0.26992 * e.omega * e.omega
                                 : 0.480 + 1.574 * e.omega - 0.176 * e.omega * e.omega;
            const double s = 1.0 + m * (1.0 - std::sqrt(e.T / tc));
            aalpha = e.a * s * s;
        }
        p.eos_aalpha[k] = (CT)aalpha;
        p.zc[k] = c.zc_A[k] != 0.0 ? 1 : 0;
        p.zcA[k] = (CT)c.zc_A[k];
        p.zc_hg[k] = (CT)(0.5 * c.G[k][k]);
        p.st_on[k] = c.st_kappa[k] != 0.0 ? 1 : 0;
        {
            const double kg = c.st_kappa[k] * c.G[k][k];
            p.st_coef[k][0] = (CT)(1.5 * c.mrt_rates[k][1] * kg);
            p.st_coef[k][1] = (CT)(-1.5 * c.mrt_rates[k][2] * kg);
            p.st_coef[k][2] = (CT)(-c.mrt_rates[k][7] * kg);
            p.st_coef[k][3] = (CT)(-c.mrt_rates[k][8] * kg);
        }
        p.wet_phi[k] = (CT)c.wet[k].phi;
        p.wet_drho[k] = (CT)c.wet[k].drho;
        p.wet_lo[k] = (CT)c.wet[k].lo;
        p.wet_hi[k] = (CT)c.wet[k].hi;
    }
    for (int a = 0; a < 3; ++a) p.body[a] = (CT)(a < h->d ? c.body_accel[a] : 0.0);
    for (int fc = 0; fc < 6; ++fc) {
        p.face_kind[fc] = h->face_kind[fc];
        for (int k = 0; k < 2; ++k) p.face_rho[fc][k] = (CT)h->face_rho[fc][k];
        for (int a = 0; a < 3; ++a) p.face_u[fc][a] = (CT)h->face_u[fc][a];
    }
    return p;
}

// ---------------------------------------------------------------- boundary preprocessing kernels
struct Geo {
    int nx, ny, nz, N;
    int periodic[3];
    int face_kind[6];
};

// link flags (integer-only): bit i = pull of direction i has no fluid source; SOLID_BIT; FACEBC_BIT
template <class L>
__global__ void k_build_flags(Geo g, const uint8_t* __restrict__ mask, uint32_t* __restrict__ flags) {
    const int id = blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= g.N) return;
    if (mask && mask[id]) { flags[id] = SOLID_BIT; return; }
    const int x = id % g.nx, t = id / g.nx, y = t % g.ny, z = t / g.ny;
    const int n[3] = {g.nx, g.ny, g.nz};
    uint32_t fl = 0;
    static_for<1, L::Q>([&](auto I) {
        constexpr int i = I;
        int pc[3] = {x - L::E[i][0], y - L::E[i][1], z - L::E[i][2]};
        int face = -1;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            if (pc[a] < 0) {
                if (g.periodic[a]) pc[a] += n[a];
                else { if (face < 0) face = 2 * a; pc[a] = 0; }
            } else if (pc[a] >= n[a]) {
                if (g.periodic[a]) pc[a] -= n[a];
                else { if (face < 0) face = 2 * a + 1; pc[a] = n[a] - 1; }
            }
        }
        if (face >= 0) {
            fl |= 1u << i;
            if (g.face_kind[face] == FACE_VELOCITY || g.face_kind[face] == FACE_PRESSURE) fl |= FACEBC_BIT;
        } else if (mask && mask[pc[0] + g.nx * (pc[1] + g.ny * pc[2])]) {
            fl |= 1u << i;
        }
    });
    flags[id] = fl;
}

// boundary solids: solid cells with >= 1 fluid neighbour under wrap/clamp indexing (R11)
template <class L>
__global__ void k_list_boundary_solids(Geo g, const uint32_t* __restrict__ flags, int* __restrict__ list, int* counter) {
    const int id = blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= g.N) return;
    if (!(flags[id] & SOLID_BIT)) return;
    const int x = id % g.nx, t = id / g.nx, y = t % g.ny, z = t / g.ny;
    const int n[3] = {g.nx, g.ny, g.nz};
    bool any = false;
    static_for<1, L::Q>([&](auto I) {
        constexpr int i = I;
        int pc[3] = {x + L::E[i][0], y + L::E[i][1], z + L::E[i][2]};
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            if (pc[a] < 0) pc[a] = g.periodic[a] ? pc[a] + n[a] : 0;
            if (pc[a] >= n[a]) pc[a] = g.periodic[a] ? pc[a] - n[a] : n[a] - 1;
        }
        if (!(flags[pc[0] + g.nx * (pc[1] + g.ny * pc[2])] & SOLID_BIT)) any = true;
    });
    if (any) list[atomicAdd(counter, 1)] = id;
}

// per boundary solid: which neighbours are fluid (same wrap/clamp indexing), so that K1b does not gather 18 flag words
template <class L>
__global__ void k_bsolid_masks(Geo g, int nb, const uint32_t* __restrict__ flags, const int* __restrict__ list, uint32_t* __restrict__ bmask) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= nb) return;
    const int id = list[b];
    const int x = id % g.nx, t = id / g.nx, y = t % g.ny, z = t / g.ny;
    const int n[3] = {g.nx, g.ny, g.nz};
    uint32_t m = 0;
    static_for<1, L::Q>([&](auto I) {
        constexpr int i = I;
        int pc[3] = {x + L::E[i][0], y + L::E[i][1], z + L::E[i][2]};
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            if (pc[a] < 0) pc[a] = g.periodic[a] ? pc[a] + n[a] : 0;
            if (pc[a] >= n[a]) pc[a] = g.periodic[a] ? pc[a] - n[a] : n[a] - 1;
        }
        if (!(flags[pc[0] + g.nx * (pc[1] + g.ny * pc[2])] & SOLID_BIT)) m |= 1u << i;
    });
    bmask[b] = m;
}

// Order in which the compaction visits the cells.  Plain: ascending cell index.  Blocked (the fluid-cell list): the
// domain is cut into bx x by x bz bricks, visited brick by brick and x-fastest inside a brick, so that the neighbours of a
// run of list entries in +-y and +-z are a few entries away in the list instead of a row or a plane of fluid cells away --
// the psi gathers and the push scatter of the compact K2 then touch a few neighbouring sectors per warp access
// (measured on config 4: scatter and gathers cost 0.45 of K2's 1.43 ms in row-major order).
struct VisitOrder {
    int nx, ny, nz, bx, by, bz, nbx, nby;   // bx = 0: plain order
    long long total;                         // positions to visit (N, or the brick-padded volume)
    __host__ __device__ int cell(long long pos) const {   // cell index at a position, -1 outside the domain
        if (bx == 0) return (int)pos;
        const int bvol = bx * by * bz;
        const long long b = pos / bvol;
        int r = (int)(pos - b * bvol);
        const int lx = r % bx; r /= bx;
        const int ly = r % by, lz = r / by;
        const int ibx = (int)(b % nbx);
        const long long t = b / nbx;
        const int iby = (int)(t % nby), ibz = (int)(t / nby);
        const int x = ibx * bx + lx, y = iby * by + ly, z = ibz * bz + lz;
        if (x >= nx || y >= ny || z >= nz) return -1;
        return x + nx * (y + ny * z);
    }
};

// Cell list by stream compaction in three small kernels: per-block counts, scan, fill.
constexpr int COMPACT_BLOCK = 1024;
__global__ void __launch_bounds__(COMPACT_BLOCK) k_fluid_count(VisitOrder vo, const uint32_t* __restrict__ flags, int* __restrict__ blockcnt,
                                                               uint32_t tmask = SOLID_BIT, uint32_t tval = 0u) {
    const long long pos = (long long)blockIdx.x * COMPACT_BLOCK + threadIdx.x;
    const int id = pos < vo.total ? vo.cell(pos) : -1;
    const int fluid = id >= 0 && (flags[id] & tmask) == tval;   // default predicate: fluid cell
    const int n = __syncthreads_count(fluid);
    if (threadIdx.x == 0) blockcnt[blockIdx.x] = n;
}
// exclusive scan of nb block counts in place (one CTA); total -> blockcnt[nb]
__global__ void __launch_bounds__(1024) k_fluid_scan(int nb, int* __restrict__ blockcnt) {
    __shared__ int part[1024];
    const int t = threadIdx.x;
    const int seg = (nb + 1023) / 1024;
    const int b0 = min(nb, t * seg), b1 = min(nb, b0 + seg);
    int s = 0;
    for (int b = b0; b < b1; ++b) s += blockcnt[b];
    part[t] = s;
    __syncthreads();
    for (int off = 1; off < 1024; off <<= 1) {
        const int v = t >= off ? part[t - off] : 0;
        __syncthreads();
        part[t] += v;
        __syncthreads();
    }
    int run = part[t] - s;
    for (int b = b0; b < b1; ++b) { const int c = blockcnt[b]; blockcnt[b] = run; run += c; }
    if (t == 1023) blockcnt[nb] = part[1023];
}
__global__ void __launch_bounds__(COMPACT_BLOCK) k_fluid_fill(VisitOrder vo, const uint32_t* __restrict__ flags, const int* __restrict__ blockoff,
                                                              int* __restrict__ list, uint32_t tmask = SOLID_BIT, uint32_t tval = 0u) {
    __shared__ int wcnt[COMPACT_BLOCK / 32];
    const long long pos = (long long)blockIdx.x * COMPACT_BLOCK + threadIdx.x;
    const int id = pos < vo.total ? vo.cell(pos) : -1;
    const int fluid = id >= 0 && (flags[id] & tmask) == tval;
    const unsigned bal = __ballot_sync(0xffffffffu, fluid);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (lane == 0) wcnt[w] = __popc(bal);
    __syncthreads();
    int off = blockoff[blockIdx.x];
    for (int k = 0; k < w; ++k) off += wcnt[k];
    if (fluid) list[off + __popc(bal & ((1u << lane) - 1u))] = id;
}

__global__ void k_mark(int n, const int* __restrict__ list, uint32_t* __restrict__ marks) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t < n) marks[list[t]] = 1u;
}

__global__ void k_export_flags(int N, const uint32_t* __restrict__ in, uint32_t* __restrict__ out) {
    const int id = blockIdx.x * blockDim.x + threadIdx.x;
    if (id < N) out[id] = in[id] & (SOLID_BIT | LINK_MASK);
}

// psi export of a component with a Zhang-Chen weight: the field holds the signed root, psi is its positive part
template <class CT>
__global__ void k_clamp0(CT* __restrict__ x, long long n) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n && x[i] < CT(0)) x[i] = CT(0);
}

// Iso-surface rendering of a resident density field (include/lbm.h: lbm_render_isosurface).  One thread per ray.
template <typename CT>
__global__ void k_render_iso(const CT* __restrict__ rho, int nx, int ny, int nz, int axis, int perx, int pery, int perz,
                             CT iso, CT* __restrict__ shade, CT* __restrict__ depth) {
    const int n[3] = {nx, ny, nz};
    const int per[3] = {perx, pery, perz};
    const long long st[3] = {1, nx, (long long)nx * ny};
    const int au = axis == 0 ? 1 : 0, av = axis == 2 ? 1 : 2, aa = axis;
    const int nu = n[au], nv = n[av], na = n[aa];
    const long long pix = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (pix >= (long long)nu * nv) return;
    const int cu = (int)(pix % nu), cv = (int)(pix / nu);
    const long long base = cu * st[au] + cv * st[av];
    // central difference along axis ax at the cell with frame coordinates (cu, cv, ck)
    auto grad = [&](int ax, int ck) -> CT {
        const int c = ax == au ? cu : (ax == av ? cv : ck);
        const int ip = per[ax] ? (c + 1 == n[ax] ? 0 : c + 1) : min(c + 1, n[ax] - 1);
        const int im = per[ax] ? (c == 0 ? n[ax] - 1 : c - 1) : max(c - 1, 0);
        const long long cell = base + ck * st[aa];
        return CT(0.5) * (rho[cell + (ip - c) * st[ax]] - rho[cell + (im - c) * st[ax]]);
    };
    CT sh = 0, dp = -1;
    CT a = rho[base];
    for (int k = 0; k + 1 < na; ++k) {
        const CT b = rho[base + (k + 1) * st[aa]];
        if ((a - iso) * (b - iso) <= CT(0) && a != b) {
            const CT w = (iso - a) / (b - a);
            const CT gu = -((CT(1) - w) * grad(au, k) + w * grad(au, k + 1));
            const CT gv = -((CT(1) - w) * grad(av, k) + w * grad(av, k + 1));
            const CT ga = -((CT(1) - w) * grad(aa, k) + w * grad(aa, k + 1));
            const CT norm = sqrt(gu * gu + gv * gv + ga * ga);
            const CT l0 = CT(0.40824829046386301637), l2 = CT(-0.81649658092772603273);   // (1, 1, -2) / sqrt(6)
            const CT dot = norm > CT(0) ? (gu * l0 + gv * l0 + ga * l2) / norm : CT(0);
            sh = CT(0.1) + CT(0.9) * (dot > CT(0) ? dot : CT(0));
            dp = CT(k) + w;
            break;
        }
        a = b;
    }
    if (shade) shade[pix] = sh;
    if (depth) depth[pix] = dp;
}

template <class TI, class TO>
__global__ void k_convert(const TI* __restrict__ in, TO* __restrict__ out, long long n) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = (TO)in[i];
}

// ---------------------------------------------------------------- helpers
int fail(lbm* h, int code, const char* what) {
    h->err = what;
    return code;
}
int cuda_fail(lbm* h, cudaError_t e, const char* where) {
    h->err = std::string(where) + ": " + cudaGetErrorString(e);
    return LBM_E_CUDA;
}
#define CU(call)                                                  \
    do {                                                          \
        cudaError_t e_ = (call);                                  \
        if (e_ != cudaSuccess) return cuda_fail(h, e_, #call);    \
    } while (0)

typedef cudaError_t (*launch_fn)(const LaunchArgs&);

launch_fn pick_launch(const lbm_config_t& c) {
    const bool d2 = c.lattice == LBM_D2Q9;
    if (c.compute_dtype == LBM_F32) {
        if (c.store_dtype == LBM_F32) return d2 ? &launch<D2Q9, float, float> : &launch<D3Q19, float, float>;
        if (c.store_dtype == LBM_F16) return d2 ? &launch<D2Q9, float, __half> : &launch<D3Q19, float, __half>;
    } else {
        if (c.store_dtype == LBM_F64) return d2 ? &launch<D2Q9, double, double> : &launch<D3Q19, double, double>;
        if (c.store_dtype == LBM_F32) return d2 ? &launch<D2Q9, double, float> : &launch<D3Q19, double, float>;
    }
    return nullptr;
}

// ---- measurement only: event brackets around hot-loop kernels
int prof_drain(lbm* h) {
    if (h->ev_pending.empty()) return LBM_OK;
    CU(cudaStreamSynchronize(h->stream));
    for (auto& pr : h->ev_pending) {
        float ms = 0.f;
        CU(cudaEventElapsedTime(&ms, pr.a, pr.b));
        h->k_ms[pr.kid] += ms;
        h->k_cnt[pr.kid] += pr.n;
        h->ev_pool.push_back(pr.a);
        h->ev_pool.push_back(pr.b);
    }
    h->ev_pending.clear();
    return LBM_OK;
}
int prof_event(lbm* h, cudaEvent_t* ev) {
    if (h->ev_pool.empty()) {
        CU(cudaEventCreate(ev));
    } else {
        *ev = h->ev_pool.back();
        h->ev_pool.pop_back();
    }
    CU(cudaEventRecord(*ev, h->stream));
    return LBM_OK;
}

int do_launch(lbm* h, int op, const void* a0, const void* a1, void* a2, int i0, int in_buf, int out_buf);

// hot-loop launch, bracketed by events while profiling is on
int hot_launch(lbm* h, int op, int kid) {
    const int i0 = op == OP_FUSED ? h->fmchunk : 0;
    if (!h->profiling) return do_launch(h, op, nullptr, nullptr, nullptr, i0, -1, -1);
    if (h->ev_pending.size() >= 2048) { int rc = prof_drain(h); if (rc) return rc; }
    lbm::EvPair pr;
    pr.kid = kid;
    pr.n = 1;
    int rc = prof_event(h, &pr.a);
    if (rc) return rc;
    rc = do_launch(h, op, nullptr, nullptr, nullptr, i0, -1, -1);
    if (rc) return rc;
    rc = prof_event(h, &pr.b);
    if (rc) return rc;
    h->ev_pending.push_back(pr);
    return LBM_OK;
}

// in_buf / out_buf: which population buffer the kernel reads / writes (-1 = current / the other one)
int do_launch(lbm* h, int op, const void* a0 = nullptr, const void* a1 = nullptr, void* a2 = nullptr, int i0 = 0,
              int in_buf = -1, int out_buf = -1);
int do_launch(lbm* h, int op, const void* a0, const void* a1, void* a2, int i0, int in_buf, int out_buf) {
    if (in_buf < 0) in_buf = h->cur;
    if (out_buf < 0) out_buf = h->cur ^ 1;
    LaunchArgs a;
    a.op = op;
    a.nc = h->cfg.n_components;
    a.coll = (h->cfg.flags & LBM_FLAG_NO_COLLIDE) ? 2 : (h->cfg.collision == LBM_MRT ? 1 : 0);
    a.bnd = h->bnd ? 1 : 0;
    a.vec = h->vec;
    const bool zc = h->cfg.zc_A[0] != 0.0 || h->cfg.st_kappa[0] != 0.0 ||
                    (h->cfg.n_components > 1 && (h->cfg.zc_A[1] != 0.0 || h->cfg.st_kappa[1] != 0.0));   // extended-force variant of K2
    a.zc = (zc && op == OP_STEP && !(h->cfg.flags & LBM_FLAG_NO_COLLIDE)) ? 1 : 0;
    a.list = (h->use_list && (op == OP_MOMENTS || (op == OP_STEP && !a.zc))) ? (h->is_compact ? 2 : 1) : 0;
    a.a0 = a0; a.a1 = a1; a.a2 = a2; a.i0 = i0;
    a.wref = h->cfg.rho_ref != 0.0 ? 1 : 0;   // (also read by the compact kernels)
    a.eq = h->feq ? (h->eq_split ? 2 + h->eq_split : (h->eq_half ? 2 : 1)) : 0;
    a.pdl = h->pdl ? 1 : 0;
    a.i1 = h->eq_ygroup;
    a.i2 = h->ws_ty;
    a.used_kernel = op == OP_FUSED ? &h->last_path : nullptr;
    a.stream = h->stream;
    launch_fn fn = pick_launch(h->cfg);
    if (!fn) return fail(h, LBM_E_UNSUPPORTED, "dtype combination not built");
    cudaError_t e;
    if (!h->params_valid) {
        if (h->cfg.compute_dtype == LBM_F32) h->pf32 = make_params<float>(h, 0, 1);
        else h->pf64 = make_params<double>(h, 0, 1);
        h->params_valid = true;
    }
    // per-launch fields
    auto patch = [&](auto& p) {
        p.f_in = h->ws + h->cv.f[in_buf];
        p.f_out = h->ws + h->cv.f[out_buf];
        p.nbsolid = h->nbsolid;
        p.bmask = h->has_bmask ? reinterpret_cast<const uint32_t*>(h->ws + h->cv.bsolid) + h->nbsolid : nullptr;
        p.nfluid = h->nfluid;
        p.nbr_stride = h->nbr_stride;
        p.cplane = h->nbr_stride;
        p.compact = h->is_compact ? 1 : 0;
        p.snbr = (h->is_compact && h->snbr_stride > 0) ? reinterpret_cast<const uint32_t*>(h->ws + h->cv.snbr) : nullptr;
        p.snbr_stride = h->snbr_stride;
        p.write_rho = (h->nbsolid > 0 || h->force_rho) ? 1 : 0;
        a.params = &p;
    };
    if (h->cfg.compute_dtype == LBM_F32) patch(h->pf32);
    else patch(h->pf64);
    e = fn(a);
    if (e != cudaSuccess) return cuda_fail(h, e, "kernel launch");
    if (!(op == OP_VIRTUAL && h->nbsolid == 0)) h->launches++;
    // k_fused_eq_split launched per chunk of planes and per group of tile rows (lbm_launch.cuh): count every launch
    if (op == OP_FUSED && a.eq >= 3 && a.i1 > 0 && h->last_path == LBM_PATH_ONE_PASS_EQ && h->fmchunk > 0) {
        const int yt = (h->cfg.ny + h->fshape.ty - 1) / h->fshape.ty;
        h->launches += (long long)((h->cfg.nz + h->fmchunk - 1) / h->fmchunk) * ((yt + a.i1 - 1) / a.i1) - 1;
    }
    return LBM_OK;
}

// FieldIO<CT> is the same layout for float and double (pointers + ints): fill it through void*
struct FieldIOAny {
    const void* in[19];
    void* out;
    long long out_stride;
    int c0, cnt;
};
static_assert(sizeof(FieldIOAny) == sizeof(FieldIO<float>) && sizeof(FieldIOAny) == sizeof(FieldIO<double>),
              "FieldIO layout");

// shape of K2F built for this configuration (mirrors the template dispatch in lbm_launch.cuh)
FusedShape fused_shape_of(const lbm_config_t& c) {
    if (c.lattice != LBM_D3Q19) return FusedShape{0, 0};
    const bool f32 = c.compute_dtype == LBM_F32;
    if (f32) return c.n_components == 1 ? fused_shape<D3Q19, float, float, 1>() : fused_shape<D3Q19, float, float, 2>();
    return c.n_components == 1 ? fused_shape<D3Q19, double, double, 1>() : fused_shape<D3Q19, double, double, 2>();
}

// Does the one-pass kernel apply, and how many planes does a CTA march?  Fully periodic, no solid cells, collision on.
void plan_fused(lbm* h) {
    h->use_fused = false;
    const lbm_config_t& c = h->cfg;
    h->feq = false;
    if (c.flags & (LBM_FLAG_TWO_PASS | LBM_FLAG_NO_COLLIDE)) return;
    if (c.zc_A[0] != 0.0 || c.st_kappa[0] != 0.0 || (c.n_components > 1 && (c.zc_A[1] != 0.0 || c.st_kappa[1] != 0.0)))
        return;   // Zhang-Chen weight / surface-tension source: two-pass path
    // D3Q19 only, rows that are whole 16-byte vectors of the storage dtype (the bulk copies carry 16-byte pads)
    if (h->bnd || h->fshape.vec == 0 || c.nx % h->fshape.vec != 0 || c.nx % (16 / (int)h->sbytes) != 0) return;
    if ((unsigned long long)c.n_components * h->q * (unsigned long long)h->plane >= (1ULL << 32)) return;   // 32-bit element offsets
    const int nm = c.nz;
    int nsm = 148, dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);   // the device the handle was created on
    // k_fused_eq: one component, BGK, tau = 1
    h->feq = c.n_components == 1 && c.collision == LBM_BGK && c.tau[0] == 1.0 && h->tune.eq != 0;
    // half-width tiles, two CTAs per SM: where a full-width last tile would leave more than a tenth of the row's lanes idle
    // and half-width tiles fewer, or where full-width tiles cannot give every SM a column (measured: 416^3 2.67 -> 2.59 ms,
    // 128^3 0.0756 -> 0.0733; 512^3 3.9 -> 4.85: full width there)
    {
        const int txf = 32 * h->fshape.vec, txh = txf / 2;
        const double uf = (double)c.nx / (((c.nx + txf - 1) / txf) * (double)txf), uh = (double)c.nx / (((c.nx + txh - 1) / txh) * (double)txh);
        const long long cols = (long long)((c.nx + txf - 1) / txf) * ((c.ny + h->fshape.ty - 1) / h->fshape.ty);
        h->eq_half = h->tune.eq_half >= 0 ? h->tune.eq_half != 0
                                          : h->fshape.vec >= 2 && ((uf < 0.9 && uh > uf + 0.05) || cols < nsm / 4);
    }
    // k_fused_eq_split (fp32 compute and storage): front / back warps per row.  Measured, ms per step, k_fused_eq (full /
    // half width) | split, late take | split, early take:   128^3 .0767 / .0733 | .0721 | .0688;  256^3 .550 | .511 | .447;
    // 320^3 1.138 | 1.074 | 1.019;  384^3 1.659 | 1.65 | 1.78;  448^3 2.980 | 2.824 | 2.749;  512^3 3.90 | 4.02 | 4.14;
    // 416^3 (paper's case) 2.714 / 2.59 | 2.491 | 2.406.  The split kernel loses where the tiles are full in x AND the
    // columns fill the GPU (384^3: 144 columns, 512^3: 256): neighbouring tiles drift apart and re-read their shared halo
    // rows from DRAM (lbm_fused_eq2.cuh) -- k_fused_eq stays there; elsewhere the split kernel with the early take runs.
    // A forced tile width (LBM_TUNE_EQ_HALF) keeps k_fused_eq.
    h->eq_split = 0;
    h->ws_ty = 0;
    h->eq_ygroup = std::max(0, h->tune.eq_ygroup);
    bool wave_launches = false;
    if (h->feq && c.compute_dtype == LBM_F32 && c.store_dtype == LBM_F32 && h->fshape.vec == 4) {
        const int txf = 32 * h->fshape.vec;
        const long long cols = (long long)((c.nx + txf - 1) / txf) * ((c.ny + h->fshape.ty - 1) / h->fshape.ty);
        const bool keep = c.nx % txf == 0 && 16 * cols >= 15LL * nsm;
        if (h->tune.eq_split >= 0) h->eq_split = std::min(h->tune.eq_split, 2);
        else if (h->tune.eq_half < 0) h->eq_split = keep ? 0 : 2;
        // ... except where those columns are ONE wave (at most one CTA per SM: 384^3, 144 columns): there the split kernel
        // with the late take wins once the march is cut into chunks of at most 192 planes that are launched one after the
        // other -- every launch starts its CTAs together and the drift between neighbouring tiles, which grows with the
        // planes marched, stays within what L2 holds.  Measured, ms per step (k_fused_eq | split late, one launch | split late,
        // a launch per chunk of 192 / 128 planes | split early, a launch per chunk): 384^3 1.659 | 1.65 | 1.540 / 1.544 | 1.73;
        // 384 x 384 x 512 2.21 | 2.23 | 2.06 (171 planes) / 2.09.  With more columns than SMs (512^3: 256) a launch per chunk
        // and per group of 32 tile rows does not pay (3.98 against 3.91 for k_fused_eq), nor with fewer columns than SMs
        // (384 x 296 x 400, 111 columns: 1.51 against 1.42 for one launch with the early take).
        wave_launches = keep && cols <= nsm && h->tune.eq_split < 0 && h->tune.eq_half < 0 && h->tune.eq_ygroup < 0 && h->tune.mchunk <= 0;
        if (wave_launches) {
            h->eq_split = 1;
            h->eq_ygroup = (c.ny + h->fshape.ty - 1) / h->fshape.ty;
        }
        if (h->eq_split) h->eq_half = false;
    }
    const bool half = h->feq && h->eq_half;
    const int tx = 32 * h->fshape.vec / (half ? 2 : 1);
    // k_fused_ws (one component) is bound by the consumers' arithmetic, one warp per tile row: where tiles of one row fewer
    // give every SM a CTA, the rows per SM and plane shrink with them (256^3, MRT: 64 columns x 2 chunks = 128 CTAs of 8 rows
    // against 74 x 2 = 148 CTAs of 7).  Chosen by  waves x (planes per chunk + 5) x rows per tile.
    h->ws_ty = 0;
    const bool eq64 = h->feq && !h->eq_split && !h->eq_half && c.compute_dtype == LBM_F64;   // k_fused_eq, fp64, full-width tiles
    if ((!h->feq && c.n_components == 1) || eq64) {
        auto best_for = [&](int t) {
            const long long tl = (long long)((c.nx + tx - 1) / tx) * ((c.ny + t - 1) / t);
            long long best = -1;
            for (int nch = 1; nch <= std::max(1, nm / 8); ++nch) {
                const int mc = (nm + nch - 1) / nch;
                const long long ctas = tl * ((nm + mc - 1) / mc);
                const long long cost = ((ctas + nsm - 1) / nsm) * (mc + 5) * t;
                if (best < 0 || cost < best) best = cost;
            }
            return best;
        };
        const int t8 = h->fshape.ty, t7 = h->fshape.ty - 1;
        if (h->tune.ws_ty >= 0) h->ws_ty = h->tune.ws_ty == t7 ? t7 : 0;
        else if (best_for(t7) < best_for(t8)) h->ws_ty = t7;
    }
    const int ty = h->ws_ty > 0 ? h->ws_ty : h->fshape.ty;
    const long long tiles = (long long)((c.nx + tx - 1) / tx) * (h->d == 3 ? (c.ny + ty - 1) / ty : 1);
    // Chunks per column of tiles: every CTA pulls two extra planes and pays a few planes' worth of pipeline fill, and
    // CTAs run in waves of one per SM, so minimise  waves * (planes per chunk + 5)  (measured on 128^3 .. 512^3: the
    // model picks 16, 128 and 128 planes, the best of the sweeps in DESIGN.md 6)
    const long long slots = (long long)nsm * (half ? 2 : 1);   // CTAs resident at a time
    long long best_cost = -1;
    int mchunk = nm;
    // ... with a ragged last x tile (k_fused_eq_split; 416 = 3.25 tiles) the CTAs are not equal -- a narrow tile moves fewer
    // bytes and finishes earlier -- and "waves" no longer describes the schedule: the launch order is then played through
    // (every CTA goes to the SM that is free first; cost of a CTA = (planes + 5) x (3/4 + 1/4 of the width fraction), the
    // weighting that ranks the sweeps below best) and the chunk with the shortest makespan wins.  With equal tiles this IS
    // waves x (planes + 5).  Measured, ms per step by planes per CTA: 416^3: 208 (the wave model's choice) 2.40, 139 2.55,
    // 104 2.35, 84 2.34, 70 2.33, 60 2.26 (picked), 52 2.30, 35 2.29;  320^3: 107 1.156, 80 1.153, 54 1.018 (picked), 40 1.045;
    // 448^3: 150 2.96, 90 2.81 (picked), 64 2.74, 56 2.77.
    const int xt_all = (c.nx + tx - 1) / tx;
    const bool ragged = h->eq_split != 0 && c.nx % tx != 0;
    const long long ycols = tiles / xt_all;
    for (int nch = 1; nch <= std::max(1, nm / 8); ++nch) {
        const int mc = (nm + nch - 1) / nch;
        const int nchunks = (nm + mc - 1) / mc;
        const long long ctas = tiles * nchunks;
        long long cost;
        if (!ragged || ctas > 200000) {
            cost = ((ctas + slots - 1) / slots) * (mc + 5);
        } else {
            std::priority_queue<long long, std::vector<long long>, std::greater<long long>> sm;
            for (long long s_ = 0; s_ < slots; ++s_) sm.push(0);
            long long makespan = 0;
            for (int z = 0; z < nchunks; ++z) {
                const long long planes = std::min(mc, nm - z * mc) + 5;
                for (long long y = 0; y < ycols; ++y)
                    for (int x = 0; x < xt_all; ++x) {
                        const long long w = std::min(tx, c.nx - x * tx);           // cells of the row the tile covers
                        const long long t = sm.top() + planes * (3 * tx + w);
                        sm.pop();
                        sm.push(t);
                        makespan = std::max(makespan, t);
                    }
            }
            cost = makespan;
        }
        if (best_cost < 0 || cost < best_cost) { best_cost = cost; mchunk = mc; }
    }
    if (wave_launches) mchunk = (nm + (nm + 191) / 192 - 1) / ((nm + 191) / 192);   // equal chunks of at most 192 planes
    if (h->tune.mchunk > 0) mchunk = std::max(1, std::min(nm, h->tune.mchunk));
    h->fmchunk = mchunk;
    // small domains cannot fill the GPU with marching CTAs: keep the two-pass path unless K2F is demanded
    const long long ctas = tiles * ((nm + mchunk - 1) / mchunk);
    // ... and rows that leave more than a fifth of the lanes of the last x tile idle (measured: 96^3, 192^3 no gain)
    const int xt = (c.nx + tx - 1) / tx;
    const bool lanes_ok = 5 * c.nx >= 4 * xt * tx;
    h->use_fused = (c.flags & LBM_FLAG_ONE_PASS) || (4 * ctas >= 3LL * nsm && lanes_ok);
}

Geo make_geo(const lbm* h) {
    Geo g;
    g.nx = h->cfg.nx; g.ny = h->cfg.ny; g.nz = h->cfg.nz; g.N = h->N;
    for (int a = 0; a < 3; ++a) g.periodic[a] = h->cfg.periodic[a] ? 1 : 0;
    for (int f = 0; f < 6; ++f) g.face_kind[f] = h->face_kind[f];
    return g;
}

// (re)build link flags and the boundary-solid list after a mask / face change
int prepare(lbm* h) {
    if (!h->dirty) return LBM_OK;
    if (h->gexec) { cudaGraphExecDestroy(h->gexec); h->gexec = nullptr; }
    h->gvalid = false;
    h->bnd = h->has_solid || !h->cfg.periodic[0] || !h->cfg.periodic[1] || (h->d == 3 && !h->cfg.periodic[2]);
    h->nbsolid = 0;
    h->nfluid = h->N;
    h->use_list = false;
    h->has_bmask = false;
    CU(cudaMemsetAsync(h->ws + h->cv.psi, 0, (size_t)h->cfg.n_components * h->N * h->cbytes, h->stream));
    CU(cudaMemsetAsync(h->ws + h->cv.rho, 0, (size_t)h->cfg.n_components * h->N * h->cbytes, h->stream));
    if (h->bnd) {
        const Geo g = make_geo(h);
        const uint8_t* mask = h->has_solid ? reinterpret_cast<const uint8_t*>(h->ws + h->cv.mask) : nullptr;
        uint32_t* flags = reinterpret_cast<uint32_t*>(h->ws + h->cv.flags);
        int* list = reinterpret_cast<int*>(h->ws + h->cv.bsolid);
        int* counter = reinterpret_cast<int*>(h->ws + h->cv.counter);
        const int block = 256, grid = (h->N + block - 1) / block;
        CU(cudaMemsetAsync(counter, 0, sizeof(int), h->stream));
        if (h->d == 2) k_build_flags<D2Q9><<<grid, block, 0, h->stream>>>(g, mask, flags);
        else k_build_flags<D3Q19><<<grid, block, 0, h->stream>>>(g, mask, flags);
        CU(cudaGetLastError());
        h->launches++;
        if (h->has_solid) {
            if (h->d == 2) k_list_boundary_solids<D2Q9><<<grid, block, 0, h->stream>>>(g, flags, list, counter);
            else k_list_boundary_solids<D3Q19><<<grid, block, 0, h->stream>>>(g, flags, list, counter);
            CU(cudaGetLastError());
            h->launches++;
            // fluid-cell list
            const int nb = (h->N + COMPACT_BLOCK - 1) / COMPACT_BLOCK;
            int* flist = reinterpret_cast<int*>(h->ws + h->cv.flist);
            int* blockcnt = flist + h->N;
            const VisitOrder plain{h->cfg.nx, h->cfg.ny, h->cfg.nz, 0, 1, 1, 1, 1, (long long)h->N};
            VisitOrder vo = plain;                      // the fluid-cell list is brick-ordered (VisitOrder)
            {
                int b[3] = {std::min(h->tune.brick[0], BRICK_MAX), std::min(h->tune.brick[1], BRICK_MAX),
                            h->cfg.nz > 1 ? std::min(h->tune.brick[2], BRICK_MAX) : 1};
                const long long vol = brick_volume(h->cfg, b);
                if (b[0] > 0 && vol < (1LL << 31)) {
                    vo.bx = b[0]; vo.by = b[1]; vo.bz = b[2];
                    vo.nbx = (h->cfg.nx + b[0] - 1) / b[0]; vo.nby = (h->cfg.ny + b[1] - 1) / b[1];
                    vo.total = vol;
                }
            }
            const int nbf = (int)((vo.total + COMPACT_BLOCK - 1) / COMPACT_BLOCK);
            k_fluid_count<<<nbf, COMPACT_BLOCK, 0, h->stream>>>(vo, flags, blockcnt);
            k_fluid_scan<<<1, 1024, 0, h->stream>>>(nbf, blockcnt);
            k_fluid_fill<<<nbf, COMPACT_BLOCK, 0, h->stream>>>(vo, flags, blockcnt, flist);
            CU(cudaGetLastError());
            h->launches += 3;
            int cnt[2] = {0, 0};
            CU(cudaMemcpyAsync(&cnt[0], counter, sizeof(int), cudaMemcpyDeviceToHost, h->stream));
            CU(cudaMemcpyAsync(&cnt[1], blockcnt + nbf, sizeof(int), cudaMemcpyDeviceToHost, h->stream));
            CU(cudaStreamSynchronize(h->stream));
            h->nbsolid = cnt[0];
            h->nfluid = cnt[1];
            if (h->nbsolid > 0) {
                // the atomic append left the boundary solids in arbitrary order: rewrite the list in the brick order of the
                // fluid list (deterministic; neighbouring threads of K1b, and the psi gathers of the compact mode, then
                // touch neighbouring memory; lbm_get_boundary_solids sorts its copy).  Scratch: the rho field (zeroed below).
                uint32_t* marks = reinterpret_cast<uint32_t*>(h->ws + h->cv.rho);
                CU(cudaMemsetAsync(marks, 0, (size_t)h->N * 4, h->stream));
                k_mark<<<(h->nbsolid + 255) / 256, 256, 0, h->stream>>>(h->nbsolid, list, marks);
                k_fluid_count<<<nbf, COMPACT_BLOCK, 0, h->stream>>>(vo, marks, blockcnt, 1u, 1u);
                k_fluid_scan<<<1, 1024, 0, h->stream>>>(nbf, blockcnt);
                k_fluid_fill<<<nbf, COMPACT_BLOCK, 0, h->stream>>>(vo, marks, blockcnt, list, 1u, 1u);
                CU(cudaGetLastError());
                h->launches += 4;
                CU(cudaMemsetAsync(h->ws + h->cv.rho, 0, (size_t)h->cfg.n_components * h->N * h->cbytes, h->stream));
                // fluid-neighbour masks behind the list (the region holds N entries)
                h->has_bmask = 2LL * h->nbsolid <= h->N;
                if (h->has_bmask) {
                    uint32_t* bm = reinterpret_cast<uint32_t*>(list + h->nbsolid);
                    if (h->d == 2) k_bsolid_masks<D2Q9><<<(h->nbsolid + 255) / 256, 256, 0, h->stream>>>(g, h->nbsolid, flags, list, bm);
                    else k_bsolid_masks<D3Q19><<<(h->nbsolid + 255) / 256, 256, 0, h->stream>>>(g, h->nbsolid, flags, list, bm);
                    CU(cudaGetLastError());
                    h->launches++;
                }
            }
            // with most cells solid the dense mapping wastes lanes and issue slots on them: one thread per fluid cell
            h->use_list = h->nfluid > 0 && h->nfluid < h->N / 2;   // (an all-solid domain has nothing to list)
            if (h->tune.list >= 0) h->use_list = h->nfluid > 0 && h->tune.list != 0;
        }
    }
    h->dirty = false;
    h->params_valid = false;
    plan_fused(h);
    // Compact mode (lbm_compact.cuh): a quarter or less of the cells fluid, plain Shan-Chen force
    const lbm_config_t& c = h->cfg;
    const bool ext_force = c.zc_A[0] != 0.0 || c.st_kappa[0] != 0.0 || (c.n_components > 1 && (c.zc_A[1] != 0.0 || c.st_kappa[1] != 0.0));
    h->compact_on = h->use_list && !ext_force && h->nfluid <= h->N / 4 && (long long)h->nfluid + h->nbsolid <= h->N &&
                    (long long)h->nfluid + h->nbsolid < (1LL << 28);   // 28-bit extended indices in the neighbour table
    if (h->tune.compact >= 0) h->compact_on = h->compact_on && h->tune.compact != 0;
    if (h->compact_on && (unsigned long long)h->q * (((unsigned long long)h->nfluid + 63) / 64 * 64) >= (1ULL << 32))
        h->compact_on = false;   // 32-bit element offsets within a component
    if (h->compact_on) {
        h->nbr_stride = ((long long)h->nfluid + 63) / 64 * 64;
        int* cmap = reinterpret_cast<int*>(h->ws + h->cv.rho);   // scratch: the rho field is rewritten before it is read
        const int* flist = reinterpret_cast<const int*>(h->ws + h->cv.flist);
        const int* bsolid = reinterpret_cast<const int*>(h->ws + h->cv.bsolid);
        CU(cudaMemsetAsync(cmap, 0xFF, (size_t)h->N * 4, h->stream));
        k_cmap_scatter<<<(h->nfluid + 255) / 256, 256, 0, h->stream>>>(h->nfluid, flist, 0, cmap);
        if (h->nbsolid > 0) k_cmap_scatter<<<(h->nbsolid + 255) / 256, 256, 0, h->stream>>>(h->nbsolid, bsolid, h->nfluid, cmap);
        CU(cudaGetLastError());
        h->launches += 2;
        int rc = do_launch(h, OP_BUILD_NBR, cmap, nullptr, h->ws + h->cv.nbr);
        if (rc) return rc;
        h->snbr_stride = 0;
        if (h->nbsolid > 0 && h->nbsolid <= h->N / 4 && !h->tune.no_snbr) {
            h->snbr_stride = ((long long)h->nbsolid + 63) / 64 * 64;
            if ((rc = do_launch(h, OP_BUILD_SNBR, cmap, nullptr, h->ws + h->cv.snbr))) return rc;
        }
        CU(cudaMemsetAsync(h->ws + h->cv.rho, 0, (size_t)c.n_components * h->N * h->cbytes, h->stream));
    }
    return LBM_OK;
}

// Bring the current population buffer into the fluid-compact (lbm_step on porous domains) or the dense layout (every
// other entry point): a gather / scatter through the other buffer.
int set_layout(lbm* h, bool compact) {
    if (!h->initialized || h->is_compact == compact) return LBM_OK;
    int rc;
    if (!compact) {
        h->is_compact = false;   // the fill below is a dense kernel
        if ((rc = do_launch(h, OP_FILL_SOLID))) return rc;
        // psi held the extended order, rho (with the boundary solids' table) the compact order: back to all-zero dense fields
        CU(cudaMemsetAsync(h->ws + h->cv.psi, 0, (size_t)h->cfg.n_components * h->N * h->cbytes, h->stream));
        CU(cudaMemsetAsync(h->ws + h->cv.rho, 0, (size_t)h->cfg.n_components * h->N * h->cbytes, h->stream));
    }
    // dense planes hold post-collision values at the writing cell, compact planes post-stream values (lbm_compact.cuh)
    if ((rc = do_launch(h, compact ? OP_PACK_C : OP_UNPACK_C))) return rc;
    h->cur ^= 1;
    h->is_compact = compact;
    return LBM_OK;
}

template <class TI, class TO>
int convert(lbm* h, const void* in, void* out, long long n) {
    const int block = 256;
    k_convert<TI, TO><<<(unsigned)((n + block - 1) / block), block, 0, h->stream>>>(static_cast<const TI*>(in),
                                                                                  static_cast<TO*>(out), n);
    CU(cudaGetLastError());
    h->launches++;
    return LBM_OK;
}

// Bring `n` values of element type `dtype` (host or device) into the compute dtype on the device.
// Returns a device pointer in *out: the source itself when no copy/convert is needed, else stage_a/stage_b.
int fetch_input(lbm* h, const void* src, long long n, int dtype, int on_device, char* stage_raw, char* stage_ct,
                const void** out) {
    const size_t eb = dtype_bytes(dtype);
    const void* dev = src;
    if (!on_device) {
        CU(cudaMemcpyAsync(stage_raw, src, (size_t)n * eb, cudaMemcpyHostToDevice, h->stream));
        dev = stage_raw;
    }
    if (dtype == h->cfg.compute_dtype) { *out = dev; return LBM_OK; }
    int rc = dtype == LBM_F32 ? convert<float, double>(h, dev, stage_ct, n) : convert<double, float>(h, dev, stage_ct, n);
    if (rc) return rc;
    *out = stage_ct;
    return LBM_OK;
}

// Deliver `n` compute-dtype values at device pointer `dev` to dst (host or device) as `dtype`.
int deliver_output(lbm* h, const void* dev, long long n, int dtype, int on_device, char* stage_conv, void* dst) {
    const void* src = dev;
    if (dtype != h->cfg.compute_dtype) {
        void* conv = on_device ? dst : stage_conv;
        int rc = dtype == LBM_F32 ? convert<double, float>(h, dev, conv, n) : convert<float, double>(h, dev, conv, n);
        if (rc) return rc;
        if (on_device) return LBM_OK;
        src = conv;
    }
    if (src != dst)
        CU(cudaMemcpyAsync(dst, src, (size_t)n * dtype_bytes(dtype),
                           on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, h->stream));
    return LBM_OK;
}

}  // namespace

// ==================================================================== C ABI
// ---- slab decomposition along the last axis: halo layers in the storage dtype, [component][direction][layer][cells of a layer]
namespace {
struct HaloGeom { long long layer, nl, chunk_bytes, plane_bytes; int rows; };
int halo_geom(lbm* h, int width, HaloGeom* g) {
    const lbm_config_t& c = h->cfg;
    g->layer = h->d == 3 ? (long long)c.nx * c.ny : (long long)c.nx;
    g->nl = h->d == 3 ? c.nz : c.ny;
    if (width < 1 || 3LL * width > g->nl) return fail(h, LBM_E_INVALID, "halo width: the last axis needs at least 3 * width layers");
    if (!c.periodic[h->d - 1]) return fail(h, LBM_E_INVALID, "halo exchange: the handle must be periodic along its last axis");
    g->chunk_bytes = (long long)width * g->layer * (long long)h->sbytes;
    g->plane_bytes = h->plane * (long long)h->sbytes;
    g->rows = c.n_components * h->q;
    return LBM_OK;
}
// copy the layers [l0, l0 + width) of every population plane to / from a packed buffer
int halo_copy(lbm* h, const HaloGeom& g, long long l0, void* packed, bool to_packed) {
    char* planes = h->ws + h->cv.f[h->cur] + l0 * g.layer * (long long)h->sbytes;
    if ((uintptr_t)packed % (uintptr_t)h->sbytes != 0) return fail(h, LBM_E_INVALID, "halo buffer alignment");
    const bool a16 = g.chunk_bytes % 16 == 0 && g.plane_bytes % 16 == 0 && ((uintptr_t)planes % 16) == 0 && ((uintptr_t)packed % 16) == 0;
    const long long unit = a16 ? 16 : (long long)h->sbytes;
    const long long ru = g.chunk_bytes / unit, pp = g.plane_bytes / unit, total = ru * g.rows;
    const unsigned blocks = (unsigned)std::min<long long>((total + 255) / 256, 148LL * 16);
    char* dst = to_packed ? static_cast<char*>(packed) : planes;
    const char* src = to_packed ? planes : static_cast<const char*>(packed);
    const long long sp = to_packed ? pp : ru, dp = to_packed ? ru : pp;
    if (unit == 16) k_halo_copy<uint4><<<blocks, 256, 0, h->stream>>>((uint4*)dst, (const uint4*)src, g.rows, ru, sp, dp);
    else if (unit == 8) k_halo_copy<uint2><<<blocks, 256, 0, h->stream>>>((uint2*)dst, (const uint2*)src, g.rows, ru, sp, dp);
    else if (unit == 4) k_halo_copy<uint32_t><<<blocks, 256, 0, h->stream>>>((uint32_t*)dst, (const uint32_t*)src, g.rows, ru, sp, dp);
    else k_halo_copy<uint16_t><<<blocks, 256, 0, h->stream>>>((uint16_t*)dst, (const uint16_t*)src, g.rows, ru, sp, dp);
    CU(cudaGetLastError());
    h->launches++;
    return LBM_OK;
}
int halo_ready(lbm* h) {
    if (!h->initialized) return fail(h, LBM_E_STATE, "halo exchange before lbm_init_fields");
    int rc = prepare(h);
    if (rc) return rc;
    return set_layout(h, false);
}
}  // namespace

// ================================================================== lbm_step_noalloc (include/lbm.h)
// One time step (S1..S7, the two-pass arrangement K1 -> K2) on caller-held populations, for callers that may not allocate
// device memory and hold no workspace: psi, the one field K1 hands to K2, lives in a file-scope device array.  Every GPU
// that loads the library holds LBM_NOALLOC_SCRATCH_BYTES of it until exit.  In host code the array's name is only a
// stand-in: the device address comes from cudaGetSymbolAddress (noalloc_scratch(), once per device) and is what the
// kernels get.  The arrays are the exported ones (post-stream f_i(x, t), compute dtype, [component][q][N]); K2 therefore
// reads its own cell and PUSHES (f_out[i][x + e_i] = f*_i(x)) where the resident kernels pull.  Same device functions
// (density, psi_of_rho, moments, psi_sums_rows, force_and_velocity, collide) in the same order as K1 / K2 of lbm_hot.cuh.
static __device__ __align__(256) unsigned char g_noalloc_scratch[LBM_NOALLOC_SCRATCH_BYTES];

template <class L, int NC, class CT>
__global__ void __launch_bounds__(256) k_noalloc_moments(const __grid_constant__ KParams<CT> p, const CT* __restrict__ f_in,
                                                         CT* __restrict__ psi) {
    for (int id = blockIdx.x * blockDim.x + threadIdx.x; id < p.N; id += gridDim.x * blockDim.x) {
#pragma unroll
        for (int k = 0; k < NC; ++k) {
            CT f[L::Q];
            static_for<0, L::Q>([&](auto I) { f[I] = f_in[((long long)k * L::Q + I) * p.N + id]; });
            psi[(long long)k * p.N + id] = psi_of_rho(p, k, density<L, CT>(f));
        }
    }
}

template <class L, int NC, class CT, int COLL>
__global__ void __launch_bounds__(256) k_noalloc_step(const __grid_constant__ KParams<CT> p, const CT* __restrict__ f_in,
                                                      const CT* __restrict__ psi, CT* __restrict__ f_out) {
    for (int id = blockIdx.x * blockDim.x + threadIdx.x; id < p.N; id += gridDim.x * blockDim.x) {
        const Cell c = make_cell<L>(p, id);
        CT f[NC][L::Q], rho[NC], j[NC][3];
#pragma unroll
        for (int k = 0; k < NC; ++k) {
            static_for<0, L::Q>([&](auto I) { f[k][I] = f_in[((long long)k * L::Q + I) * p.N + id]; });
            moments<L, CT>(f[k], rho[k], j[k]);
        }
        CT u[3] = {CT(0), CT(0), CT(0)}, du[NC][3], S[NC][3], pc[NC];
#pragma unroll
        for (int kp = 0; kp < NC; ++kp) {
            const CT* ps = psi + (long long)kp * p.N + id;
            auto rowfn = [&](auto DY, auto DZ, auto NX, CT (&t)[1], CT& left, CT& right) {
                constexpr int dy = DY, dz = DZ;
                t[0] = ps[nbr_offset<0, dy, dz>(c)];
                if constexpr (NX != 0) {
                    left = ps[nbr_offset<-1, dy, dz>(c)];
                    right = ps[nbr_offset<1, dy, dz>(c)];
                }
            };
            CT S1[3][1], pc1[1];
            psi_sums_rows<L, CT, 1>(rowfn, S1, pc1);
            S[kp][0] = S1[0][0]; S[kp][1] = S1[1][0]; S[kp][2] = S1[2][0];
            pc[kp] = pc1[0];
        }
        force_and_velocity<NC, CT>(p, rho, j, S, pc, u, du);
#pragma unroll
        for (int k = 0; k < NC; ++k) {
            collide<L, COLL, CT>(p, k, rho[k], u, du[k], f[k]);
            CT* out = f_out + (long long)k * L::Q * p.N + id;
            static_for<0, L::Q>([&](auto I) {
                out[(long long)I * p.N + nbr_offset<L::E[I][0], L::E[I][1], L::E[I][2]>(c)] = f[k][I];
            });
        }
    }
}

namespace {
thread_local std::string g_noalloc_err;
int noalloc_fail(int code, const std::string& what) {
    g_noalloc_err = what;
    return code;
}
// device address of the static scratch array on the CURRENT device, looked up once per device
int noalloc_scratch(void** out) {
    static std::mutex mu;
    static void* ptr[64] = {nullptr};
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return noalloc_fail(LBM_E_CUDA, std::string("cudaGetDevice: ") + cudaGetErrorString(e));
    if (dev < 0 || dev >= 64) return noalloc_fail(LBM_E_UNSUPPORTED, "lbm_step_noalloc: device ordinal beyond 63");
    std::lock_guard<std::mutex> lock(mu);
    if (!ptr[dev]) {
        void* q = nullptr;
        e = cudaGetSymbolAddress(&q, g_noalloc_scratch);
        if (e != cudaSuccess || !q) {
            cudaGetLastError();
            return noalloc_fail(LBM_E_CUDA, std::string("cudaGetSymbolAddress(g_noalloc_scratch): ") + cudaGetErrorString(e));
        }
        ptr[dev] = q;
    }
    *out = ptr[dev];
    return LBM_OK;
}

template <class L, int NC, class CT, int COLL>
cudaError_t noalloc_launch(const KParams<CT>& p, const void* f_in, void* scratch, void* f_out, cudaStream_t stream) {
    const unsigned blocks = (unsigned)std::min<long long>(((long long)p.N + 255) / 256, 148LL * 32);
    k_noalloc_moments<L, NC, CT><<<blocks, 256, 0, stream>>>(p, static_cast<const CT*>(f_in), static_cast<CT*>(scratch));
    k_noalloc_step<L, NC, CT, COLL><<<blocks, 256, 0, stream>>>(p, static_cast<const CT*>(f_in), static_cast<const CT*>(scratch),
                                                              static_cast<CT*>(f_out));
    return cudaGetLastError();
}
template <class CT>
cudaError_t noalloc_dispatch(const lbm_config_t& c, const KParams<CT>& p, const void* f_in, void* scratch, void* f_out,
                             cudaStream_t stream) {
    auto with_l = [&](auto Ltag, auto NC, auto COLL) {
        using L = decltype(Ltag);
        return noalloc_launch<L, NC, CT, COLL>(p, f_in, scratch, f_out, stream);
    };
    auto with_nc = [&](auto Ltag, auto COLL) {
        return c.n_components == 1 ? with_l(Ltag, IC<1>{}, COLL) : with_l(Ltag, IC<2>{}, COLL);
    };
    auto with_coll = [&](auto Ltag) { return c.collision == LBM_MRT ? with_nc(Ltag, IC<1>{}) : with_nc(Ltag, IC<0>{}); };
    return c.lattice == LBM_D2Q9 ? with_coll(D2Q9{}) : with_coll(D3Q19{});
}
}  // namespace

extern "C" {

size_t lbm_workspace_bytes(const lbm_config_t* cfg) {
    if (check_config(cfg) != LBM_OK) return 0;
    return carve(*cfg).total;
}

int lbm_create(const lbm_config_t* cfg, void* d_workspace, size_t workspace_bytes, lbm_stream_t stream, lbm_t** out) {
    if (!out) return LBM_E_INVALID;
    *out = nullptr;
    int rc = check_config(cfg);
    if (rc != LBM_OK) return rc;
    if (!pick_launch(*cfg)) return LBM_E_UNSUPPORTED;
    const Carve cv = carve(*cfg);
    if (!d_workspace || workspace_bytes < cv.total || (reinterpret_cast<uintptr_t>(d_workspace) % ALIGN) != 0)
        return LBM_E_NOMEM;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return LBM_E_CUDA;  // no CPU fallback
    cudaPointerAttributes attr;
    if (cudaPointerGetAttributes(&attr, d_workspace) != cudaSuccess || attr.type != cudaMemoryTypeDevice) {
        cudaGetLastError();
        return LBM_E_INVALID;
    }
    lbm* h = new (std::nothrow) lbm();
    if (!h) return LBM_E_NOMEM;
    h->cfg = *cfg;
    h->q = q_of(cfg->lattice);
    h->d = cfg->lattice == LBM_D2Q9 ? 2 : 3;
    h->N = cfg->nx * cfg->ny * cfg->nz;
    h->plane = ((long long)h->N + 63) / 64 * 64;
    h->sbytes = dtype_bytes(cfg->store_dtype);
    h->cbytes = dtype_bytes(cfg->compute_dtype);
    h->stream = static_cast<cudaStream_t>(stream);
    h->ws = static_cast<char*>(d_workspace);
    h->cv = cv;
    h->cur = 0;
    h->vec = 1;
    {   // widest vector the hot kernels were built with for this dtype / component count, if nx allows it
        const int sb = (int)h->sbytes, cb = (int)h->cbytes;
        int v = 16 / sb;
        const int cap = 4 / (cfg->n_components * (cb / 4));
        if (v > cap) v = cap;
        if (v < 1) v = 1;
        if (cfg->nx % v == 0) h->vec = v;
    }
    h->params_valid = false;
    h->tune = Tune::from_env();
    h->fshape = fused_shape_of(*cfg);
    h->fmchunk = 1;
    h->use_fused = false;
    h->feq = false;
    h->eq_half = false;
    h->eq_split = 0;
    h->last_path = LBM_PATH_NONE;
    h->gexec = nullptr;
    h->gcur = 0;
    h->glaunches = 0;
    h->gvalid = false;
    h->gfailed = false;
    h->coop_failed = false;
    h->tile_failed = false;
    h->initialized = false;
    h->has_solid = false;
    h->dirty = true;
    h->bnd = false;
    h->force_rho = false;
    h->nbsolid = 0;
    h->nfluid = h->N;
    h->pdl = false;
    h->has_bmask = false;
    h->compact_on = false;
    h->is_compact = false;
    h->nbr_stride = 0;
    h->snbr_stride = 0;
    h->use_list = false;
    h->steps = 0;
    h->launches = 0;
    h->profiling = false;
    for (int k = 0; k < LBM_K_COUNT; ++k) { h->k_ms[k] = 0.0; h->k_cnt[k] = 0; }
    for (int f = 0; f < 6; ++f) {
        h->face_kind[f] = cfg->periodic[f / 2] ? LBM_FACE_PERIODIC : LBM_FACE_WALL;
        h->face_rho[f][0] = h->face_rho[f][1] = 1.0;
        h->face_u[f][0] = h->face_u[f][1] = h->face_u[f][2] = 0.0;
    }
    *out = h;
    return LBM_OK;
}

void lbm_destroy(lbm_t* h) {
    if (!h) return;
    for (auto& pr : h->ev_pending) { cudaEventDestroy(pr.a); cudaEventDestroy(pr.b); }
    for (auto e : h->ev_pool) cudaEventDestroy(e);
    if (h->gexec) cudaGraphExecDestroy(h->gexec);
    delete h;
}

int lbm_set_profiling(lbm_t* h, int enable) {
    if (!h) return LBM_E_INVALID;
    if (!enable) { int rc = prof_drain(h); if (rc) return rc; }
    h->profiling = enable != 0;
    return LBM_OK;
}

int lbm_get_kernel_times(lbm_t* h, double* ms_total, int64_t* launches) {
    if (!h) return LBM_E_INVALID;
    int rc = prof_drain(h);
    if (rc) return rc;
    for (int k = 0; k < LBM_K_COUNT; ++k) {
        if (ms_total) ms_total[k] = h->k_ms[k];
        if (launches) launches[k] = h->k_cnt[k];
        h->k_ms[k] = 0.0;
        h->k_cnt[k] = 0;
    }
    return LBM_OK;
}

int lbm_set_solid_mask(lbm_t* h, const uint8_t* mask, int on_device) {
    if (!h || !mask) return LBM_E_INVALID;
    if (h->initialized) return fail(h, LBM_E_STATE, "lbm_set_solid_mask must precede lbm_init_fields");
    CU(cudaMemcpyAsync(h->ws + h->cv.mask, mask, (size_t)h->N,
                       on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, h->stream));
    if (!on_device) CU(cudaStreamSynchronize(h->stream));
    h->has_solid = true;
    h->dirty = true;
    return LBM_OK;
}

int lbm_set_face_bc(lbm_t* h, int face, int kind, const double* rho_w, const double* u_w) {
    if (!h) return LBM_E_INVALID;
    if (face < 0 || face >= 2 * h->d) return fail(h, LBM_E_INVALID, "face out of range");
    if (h->cfg.periodic[face / 2]) return fail(h, LBM_E_INVALID, "face belongs to a periodic axis");
    if (kind != LBM_FACE_WALL && kind != LBM_FACE_VELOCITY && kind != LBM_FACE_PRESSURE)
        return fail(h, LBM_E_INVALID, "face kind");
    // the stored planes already hold the face rule of the step before (it is applied at the writing cell): a change
    // between steps would take effect one step late, so it is only accepted before the first step
    if (h->initialized && h->steps > 0) return fail(h, LBM_E_STATE, "lbm_set_face_bc after lbm_step: call lbm_init_fields first");
    h->face_kind[face] = kind;
    for (int k = 0; k < 2; ++k) h->face_rho[face][k] = rho_w ? rho_w[k] : 1.0;
    for (int a = 0; a < 3; ++a) h->face_u[face][a] = u_w ? u_w[a] : 0.0;
    h->dirty = true;
    return LBM_OK;
}

int lbm_init_fields(lbm_t* h, const void* const* rho, const void* u, int dtype, int on_device) {
    if (!h || !rho) return LBM_E_INVALID;
    if (dtype != LBM_F32 && dtype != LBM_F64) return fail(h, LBM_E_INVALID, "dtype");
    int rc = prepare(h);
    if (rc) return rc;
    h->is_compact = false;   // whatever the buffers held is overwritten in the dense layout
    const int nc = h->cfg.n_components;
    for (int k = 0; k < nc; ++k)
        if (!rho[k]) return fail(h, LBM_E_INVALID, "rho[k] is NULL");
    const size_t eb = dtype_bytes(dtype);
    const int chunk = std::min(h->N, CHUNK_CELLS);
    for (int c0 = 0; c0 < h->N; c0 += chunk) {
        const int cnt = std::min(chunk, h->N - c0);
        FieldIOAny io;
        std::memset(&io, 0, sizeof io);
        io.c0 = c0;
        io.cnt = cnt;
        // slot s of the staging areas: raw bytes in stage_a, compute-dtype values in stage_b
        auto stage = [&](int slot, const void* src, const void** dev) {
            return fetch_input(h, src, cnt, dtype, on_device, h->ws + h->cv.stage_a + (size_t)slot * chunk * 8,
                               h->ws + h->cv.stage_b + (size_t)slot * chunk * 8, dev);
        };
        for (int k = 0; k < nc; ++k)
            if ((rc = stage(k, static_cast<const char*>(rho[k]) + (size_t)c0 * eb, &io.in[k]))) return rc;
        if (u)
            for (int a = 0; a < h->d; ++a)
                if ((rc = stage(2 + a, static_cast<const char*>(u) + ((size_t)a * h->N + c0) * eb, &io.in[2 + a])))
                    return rc;
        // post-stream f(x,0) into BOTH buffers
        rc = do_launch(h, OP_INIT, &io, nullptr, h->ws + h->cv.f[h->cur ^ 1], h->bnd ? 1 : 0, h->cur ^ 1, h->cur);
        if (rc) return rc;
        if (!on_device) CU(cudaStreamSynchronize(h->stream));  // staging slots are reused by the next chunk
    }
    // scatter into the storage convention of the hot loop: read buffer cur^1, write buffer cur
    if ((rc = do_launch(h, OP_UNSTREAM, nullptr, nullptr, nullptr, -1, h->cur ^ 1, h->cur))) return rc;
    h->steps = 0;
    h->initialized = true;
    return LBM_OK;
}

int lbm_step(lbm_t* h, int n) {
    if (!h || n < 0) return LBM_E_INVALID;
    if (!h->initialized) return fail(h, LBM_E_STATE, "lbm_step before lbm_init_fields");
    int rc = prepare(h);
    if (rc) return rc;
    if ((rc = set_layout(h, h->compact_on))) return rc;
    if ((h->cfg.flags & LBM_FLAG_ONE_PASS) && !h->use_fused)
        return fail(h, LBM_E_UNSUPPORTED, "LBM_FLAG_ONE_PASS: the one-pass kernel does not apply to this configuration");
    // one time step: K2F, or K1 (+K1b) + K2
    auto step_once = [&]() -> int {
        int r;
        if (h->use_fused) {
            if ((r = hot_launch(h, OP_FUSED, LBM_K_FUSED))) return r;
        } else {
            if (!(h->cfg.flags & LBM_FLAG_NO_COLLIDE)) {
                if ((r = hot_launch(h, OP_MOMENTS, LBM_K_MOMENTS))) return r;
                if (h->nbsolid > 0 && (r = hot_launch(h, OP_VIRTUAL, LBM_K_VIRTUAL))) return r;
            }
            if ((r = hot_launch(h, OP_STEP, LBM_K_STEP))) return r;
            h->last_path = h->is_compact ? LBM_PATH_TWO_PASS_COMPACT : LBM_PATH_TWO_PASS;
        }
        h->cur ^= 1;
        h->steps++;
        return LBM_OK;
    };
    // Small domains are bound by kernel launches (a D2Q9 64 x 64 step is two ~3 us kernels).  First choice: ONE persistent
    // kernel for all n steps (lbm_small.cuh: resident CTAs, grid barriers between the phases).  Where the cooperative launch
    // is not available: GRAPH_STEPS steps are captured once into a CUDA graph and replayed.  Not while profiling (event brackets), not on a stream that cannot
    // be captured (the legacy default stream): then, and for large domains, the kernels are launched one by one.
    constexpr int GRAPH_STEPS = 16;   // even: the ping-pong parity is the same after a replay
    const bool small = (long long)h->N * h->cfg.n_components <= (1LL << 22);
    // ... and each kernel is launched as a programmatic dependent of the one before it (pdl_begin), which hides most of
    // the launch latency between them
    const bool ext_force = h->cfg.zc_A[0] != 0.0 || h->cfg.st_kappa[0] != 0.0 ||
                           (h->cfg.n_components > 1 && (h->cfg.zc_A[1] != 0.0 || h->cfg.st_kappa[1] != 0.0));
    // (while profiling, a persistent launch is bracketed as a whole and counted as n steps of LBM_K_PERSISTENT)
    auto persistent_launch = [&](int op, unsigned* ctr) -> int {
        lbm::EvPair pr;
        pr.kid = LBM_K_PERSISTENT;
        pr.n = n;
        int r;
        if (h->profiling && (r = prof_event(h, &pr.a))) return r;
        r = do_launch(h, op, nullptr, nullptr, ctr, n);
        if (r != LBM_OK) {
            if (h->profiling) h->ev_pool.push_back(pr.a);
            return r;
        }
        if (h->profiling) {
            if ((r = prof_event(h, &pr.b))) return r;
            h->ev_pending.push_back(pr);
        }
        return LBM_OK;
    };
    if (small && n >= 2 && h->d == 2 && !h->tile_failed && !h->tune.no_coop && !h->tune.no_tile && !h->use_fused &&
        !h->use_list && !ext_force && !(h->cfg.flags & LBM_FLAG_NO_COLLIDE)) {
        // 2-D: rho / psi recomputed on a ring around each CTA's tile, ONE grid barrier per step (k_steps_tile)
        unsigned* ctr = reinterpret_cast<unsigned*>(h->ws + h->cv.counter + 64);
        CU(cudaMemsetAsync(ctr, 0, sizeof(unsigned), h->stream));
        rc = persistent_launch(OP_TILE, ctr);
        if (rc == LBM_OK) {
            h->cur ^= (n & 1);
            h->steps += n;
            h->last_path = LBM_PATH_ONE_PASS_TILE;
            return LBM_OK;
        }
        h->tile_failed = true;
        h->err.clear();
    }
    if (small && n >= 2 && !h->coop_failed && !h->tune.no_coop && !h->use_fused && !h->use_list && !ext_force) {
        unsigned* ctr = reinterpret_cast<unsigned*>(h->ws + h->cv.counter + 64);
        CU(cudaMemsetAsync(ctr, 0, sizeof(unsigned), h->stream));
        rc = persistent_launch(OP_COOP, ctr);
        if (rc == LBM_OK) {
            h->cur ^= (n & 1);
            h->steps += n;
            h->last_path = LBM_PATH_TWO_PASS_PERSISTENT;
            return LBM_OK;
        }
        h->coop_failed = true;   // not available / more cells than resident threads: the graph or plain launches below
        h->err.clear();
    }
    struct PdlScope { lbm* h; ~PdlScope() { h->pdl = false; } } pdl_scope{h};
    h->pdl = small && !h->profiling && !h->tune.no_pdl;
    if (small && !h->profiling && !h->gfailed && n >= 2 * GRAPH_STEPS + 1 && !h->tune.no_graph) {
        if ((rc = step_once())) return rc;      // first step plainly: one-time kernel attribute set-up happens outside capture
        --n;
        if (!h->gvalid) {
            const int cur0 = h->cur, path0 = h->last_path;
            const int64_t steps0 = h->steps, launches0 = h->launches;
            cudaGraph_t graph = nullptr;
            bool ok = cudaStreamBeginCapture(h->stream, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
            if (ok) {
                for (int s = 0; s < GRAPH_STEPS && ok; ++s) ok = step_once() == LBM_OK;
                ok = (cudaStreamEndCapture(h->stream, &graph) == cudaSuccess) && ok && graph != nullptr;
            }
            if (ok) ok = cudaGraphInstantiate(&h->gexec, graph, 0) == cudaSuccess;
            if (graph) cudaGraphDestroy(graph);
            h->glaunches = h->launches - launches0;
            h->cur = cur0; h->steps = steps0; h->launches = launches0; h->last_path = path0;   // nothing ran yet
            if (ok) { h->gvalid = true; h->gcur = cur0; }
            else { cudaGetLastError(); h->gfailed = true; h->gexec = nullptr; }
        }
        if (h->gvalid) {
            if (h->cur != h->gcur) { if ((rc = step_once())) return rc; --n; }
            while (n >= GRAPH_STEPS) {
                CU(cudaGraphLaunch(h->gexec, h->stream));
                h->steps += GRAPH_STEPS;
                h->launches += h->glaunches;
                n -= GRAPH_STEPS;
            }
        }
    }
    for (int s = 0; s < n; ++s)
        if ((rc = step_once())) return rc;
    return LBM_OK;
}

int lbm_render_isosurface(lbm_t* h, int comp, double iso, int axis, void* shade, void* depth, int dtype, int on_device) {
    if (!h || (!shade && !depth)) return LBM_E_INVALID;
    if (comp < 0 || comp >= h->cfg.n_components) return fail(h, LBM_E_INVALID, "component");
    if (axis < 0 || axis > 2) return fail(h, LBM_E_INVALID, "axis");
    if (dtype != LBM_F32 && dtype != LBM_F64) return fail(h, LBM_E_INVALID, "dtype");
    if (!h->initialized) return fail(h, LBM_E_STATE, "lbm_render_isosurface before lbm_init_fields");
    int rc = prepare(h);
    if (rc) return rc;
    if ((rc = set_layout(h, false))) return rc;
    h->force_rho = true;
    rc = do_launch(h, OP_MOMENTS);
    h->force_rho = false;
    if (rc) return rc;
    if (h->nbsolid > 0 && (rc = do_launch(h, OP_VIRTUAL))) return rc;
    const lbm_config_t& c = h->cfg;
    const int dims[3] = {c.nx, c.ny, c.nz};
    const long long npix = (long long)h->N / dims[axis];
    // the images go to the free population buffer (2 fields of at most N values)
    char* scratch = h->ws + h->cv.f[h->cur ^ 1];
    char* sh_dev = scratch;
    char* dp_dev = scratch + (size_t)npix * h->cbytes;
    const char* field = h->ws + h->cv.rho + (size_t)comp * h->N * h->cbytes;
    const unsigned grid = (unsigned)((npix + 127) / 128);
    if (c.compute_dtype == LBM_F32)
        k_render_iso<float><<<grid, 128, 0, h->stream>>>(reinterpret_cast<const float*>(field), c.nx, c.ny, c.nz, axis,
                                                         c.periodic[0], c.periodic[1], c.periodic[2], (float)iso,
                                                         reinterpret_cast<float*>(sh_dev), reinterpret_cast<float*>(dp_dev));
    else
        k_render_iso<double><<<grid, 128, 0, h->stream>>>(reinterpret_cast<const double*>(field), c.nx, c.ny, c.nz, axis,
                                                          c.periodic[0], c.periodic[1], c.periodic[2], iso,
                                                          reinterpret_cast<double*>(sh_dev), reinterpret_cast<double*>(dp_dev));
    CU(cudaGetLastError());
    h->launches++;
    const size_t eb = dtype_bytes(dtype);
    const long long chunk = std::min<long long>(npix, CHUNK_CELLS);
    auto deliver_image = [&](const char* dev, void* dst) -> int {
        for (long long c0 = 0; c0 < npix; c0 += chunk) {
            const long long cnt = std::min(chunk, npix - c0);
            int r = deliver_output(h, dev + (size_t)c0 * h->cbytes, cnt, dtype, on_device, h->ws + h->cv.stage_a,
                                   static_cast<char*>(dst) + (size_t)c0 * eb);
            if (r) return r;
            if (!on_device && dtype != h->cfg.compute_dtype) CU(cudaStreamSynchronize(h->stream));
        }
        return LBM_OK;
    };
    if (shade && (rc = deliver_image(sh_dev, shade))) return rc;
    if (depth && (rc = deliver_image(dp_dev, depth))) return rc;
    if (!on_device) CU(cudaStreamSynchronize(h->stream));
    return LBM_OK;
}

int lbm_get_macroscopic(lbm_t* h, void* const* rho, void* u, void* p, int dtype, int on_device) {
    if (!h) return LBM_E_INVALID;
    if (dtype != LBM_F32 && dtype != LBM_F64) return fail(h, LBM_E_INVALID, "dtype");
    if (!h->initialized) return fail(h, LBM_E_STATE, "lbm_get_macroscopic before lbm_init_fields");
    int rc = prepare(h);
    if (rc) return rc;
    if ((rc = set_layout(h, false))) return rc;
    const int nc = h->cfg.n_components;
    // refresh rho / psi of the current state: K1 (with rho output) and K1b
    h->force_rho = true;
    rc = do_launch(h, OP_MOMENTS);
    h->force_rho = false;
    if (rc) return rc;
    if (h->nbsolid > 0 && (rc = do_launch(h, OP_VIRTUAL))) return rc;
    // u and p go to the free population buffer ((d+1) compute-dtype fields always fit in q planes)
    char* scratch = h->ws + h->cv.f[h->cur ^ 1];
    char* u_dev = scratch;
    char* p_dev = scratch + (size_t)h->d * h->N * h->cbytes;
    if (u || p) {
        rc = do_launch(h, OP_EXPORT_MACRO, u ? u_dev : nullptr, p ? p_dev : nullptr);
        if (rc) return rc;
    }
    const size_t eb = dtype_bytes(dtype);
    const int chunk = std::min(h->N, CHUNK_CELLS);
    auto deliver_field = [&](const char* dev, void* dst) -> int {
        for (int c0 = 0; c0 < h->N; c0 += chunk) {
            const int cnt = std::min(chunk, h->N - c0);
            int r = deliver_output(h, dev + (size_t)c0 * h->cbytes, cnt, dtype, on_device, h->ws + h->cv.stage_a,
                                   static_cast<char*>(dst) + (size_t)c0 * eb);
            if (r) return r;
            if (!on_device && dtype != h->cfg.compute_dtype) CU(cudaStreamSynchronize(h->stream));
        }
        return LBM_OK;
    };
    if (rho)
        for (int k = 0; k < nc; ++k)
            if (rho[k] && (rc = deliver_field(h->ws + h->cv.rho + (size_t)k * h->N * h->cbytes, rho[k]))) return rc;
    if (u)
        for (int a = 0; a < h->d; ++a)
            if ((rc = deliver_field(u_dev + (size_t)a * h->N * h->cbytes, static_cast<char*>(u) + (size_t)a * h->N * eb)))
                return rc;
    if (p && (rc = deliver_field(p_dev, p))) return rc;
    if (!on_device) CU(cudaStreamSynchronize(h->stream));
    return LBM_OK;
}

int lbm_get_populations(lbm_t* h, int comp, void* f, int dtype, int on_device) {
    if (!h || !f) return LBM_E_INVALID;
    if (comp < 0 || comp >= h->cfg.n_components) return fail(h, LBM_E_INVALID, "component");
    if (dtype != LBM_F32 && dtype != LBM_F64) return fail(h, LBM_E_INVALID, "dtype");
    if (!h->initialized) return fail(h, LBM_E_STATE, "lbm_get_populations before lbm_init_fields");
    int rc = prepare(h);
    if (rc) return rc;
    if ((rc = set_layout(h, false))) return rc;
    const size_t eb = dtype_bytes(dtype);
    if (on_device && dtype == h->cfg.compute_dtype) {  // straight into the caller's array
        FieldIOAny io;
        std::memset(&io, 0, sizeof io);
        io.out = f; io.out_stride = h->N; io.c0 = 0; io.cnt = h->N;
        return do_launch(h, OP_EXPORT_POP, &io, nullptr, nullptr, comp);
    }
    const int chunk = std::min(h->N, CHUNK_CELLS);
    for (int c0 = 0; c0 < h->N; c0 += chunk) {
        const int cnt = std::min(chunk, h->N - c0);
        FieldIOAny io;
        std::memset(&io, 0, sizeof io);
        io.out = h->ws + h->cv.stage_b; io.out_stride = cnt; io.c0 = c0; io.cnt = cnt;
        if ((rc = do_launch(h, OP_EXPORT_POP, &io, nullptr, nullptr, comp))) return rc;
        for (int i = 0; i < h->q; ++i) {
            rc = deliver_output(h, h->ws + h->cv.stage_b + (size_t)i * cnt * h->cbytes, cnt, dtype, on_device,
                                h->ws + h->cv.stage_a + (size_t)i * chunk * 8,
                                static_cast<char*>(f) + ((size_t)i * h->N + c0) * eb);
            if (rc) return rc;
        }
        if (!on_device) CU(cudaStreamSynchronize(h->stream));
    }
    return LBM_OK;
}

int lbm_set_populations(lbm_t* h, int comp, const void* f, int dtype, int on_device) {
    if (!h || !f) return LBM_E_INVALID;
    if (comp < 0 || comp >= h->cfg.n_components) return fail(h, LBM_E_INVALID, "component");
    if (dtype != LBM_F32 && dtype != LBM_F64) return fail(h, LBM_E_INVALID, "dtype");
    if (!h->initialized) return fail(h, LBM_E_STATE, "lbm_set_populations before lbm_init_fields");
    if (h->steps != 0) return fail(h, LBM_E_STATE, "lbm_set_populations is only valid right after lbm_init_fields");
    int rc = prepare(h);
    if (rc) return rc;
    if ((rc = set_layout(h, false))) return rc;
    const size_t eb = dtype_bytes(dtype);
    const int chunk = std::min(h->N, CHUNK_CELLS);
    for (int c0 = 0; c0 < h->N; c0 += chunk) {
        const int cnt = std::min(chunk, h->N - c0);
        FieldIOAny io;
        std::memset(&io, 0, sizeof io);
        io.c0 = c0; io.cnt = cnt;
        for (int i = 0; i < h->q; ++i) {
            rc = fetch_input(h, static_cast<const char*>(f) + ((size_t)i * h->N + c0) * eb, cnt, dtype, on_device,
                             h->ws + h->cv.stage_a + (size_t)i * chunk * 8, h->ws + h->cv.stage_b + (size_t)i * chunk * 8,
                             &io.in[i]);
            if (rc) return rc;
        }
        rc = do_launch(h, OP_IMPORT_POP, &io, nullptr, h->ws + h->cv.f[h->cur ^ 1], comp, h->cur ^ 1, h->cur);
        if (rc) return rc;
        if (!on_device) CU(cudaStreamSynchronize(h->stream));
    }
    // both buffers now hold the post-stream values of this component: scatter cur^1 -> cur (storage convention)
    return do_launch(h, OP_UNSTREAM, nullptr, nullptr, nullptr, comp, h->cur ^ 1, h->cur);
}

int lbm_get_link_flags(lbm_t* h, uint32_t* flags, int on_device) {
    if (!h || !flags) return LBM_E_INVALID;
    int rc = prepare(h);
    if (rc) return rc;
    uint32_t* tmp = reinterpret_cast<uint32_t*>(h->ws + h->cv.f[h->cur ^ 1]);
    if (!h->bnd) {
        CU(cudaMemsetAsync(on_device ? (void*)flags : (void*)tmp, 0, (size_t)h->N * 4, h->stream));
    } else {
        const int block = 256;
        k_export_flags<<<(h->N + block - 1) / block, block, 0, h->stream>>>(
            h->N, reinterpret_cast<const uint32_t*>(h->ws + h->cv.flags), on_device ? flags : tmp);
        CU(cudaGetLastError());
        h->launches++;
    }
    if (!on_device) {
        CU(cudaMemcpyAsync(flags, tmp, (size_t)h->N * 4, cudaMemcpyDeviceToHost, h->stream));
        CU(cudaStreamSynchronize(h->stream));
    }
    return LBM_OK;
}

int64_t lbm_get_boundary_solids(lbm_t* h, int64_t* out, int64_t capacity) {
    if (!h) return LBM_E_INVALID;
    int rc = prepare(h);
    if (rc) return rc;
    if (!out || h->nbsolid == 0) return h->nbsolid;
    std::vector<int> tmp((size_t)h->nbsolid);
    cudaError_t e = cudaMemcpyAsync(tmp.data(), h->ws + h->cv.bsolid, (size_t)h->nbsolid * 4, cudaMemcpyDeviceToHost,
                                    h->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
    if (e != cudaSuccess) return cuda_fail(h, e, "boundary solid readback");
    std::sort(tmp.begin(), tmp.end());   // the device list is in the brick order of the fluid list
    for (int64_t b = 0; b < h->nbsolid && b < capacity; ++b) out[b] = tmp[(size_t)b];
    return h->nbsolid;
}

int lbm_get_psi(lbm_t* h, int comp, void* psi, int dtype, int on_device) {
    if (!h || !psi) return LBM_E_INVALID;
    if (comp < 0 || comp >= h->cfg.n_components) return fail(h, LBM_E_INVALID, "component");
    if (dtype != LBM_F32 && dtype != LBM_F64) return fail(h, LBM_E_INVALID, "dtype");
    if (!h->initialized) return fail(h, LBM_E_STATE, "lbm_get_psi before lbm_init_fields");
    int rc = prepare(h);
    if (rc) return rc;
    if ((rc = set_layout(h, false))) return rc;
    if ((rc = do_launch(h, OP_MOMENTS))) return rc;
    if (h->nbsolid > 0 && (rc = do_launch(h, OP_VIRTUAL))) return rc;
    if (h->cfg.zc_A[comp] != 0.0) {   // the next lbm_step recomputes the field anyway
        char* field = h->ws + h->cv.psi + (size_t)comp * h->N * h->cbytes;
        const unsigned grid = (unsigned)((h->N + 255) / 256);
        if (h->cfg.compute_dtype == LBM_F32) k_clamp0<float><<<grid, 256, 0, h->stream>>>(reinterpret_cast<float*>(field), h->N);
        else k_clamp0<double><<<grid, 256, 0, h->stream>>>(reinterpret_cast<double*>(field), h->N);
        CU(cudaGetLastError());
        h->launches++;
    }
    const size_t eb = dtype_bytes(dtype);
    const int chunk = std::min(h->N, CHUNK_CELLS);
    const char* dev = h->ws + h->cv.psi + (size_t)comp * h->N * h->cbytes;
    for (int c0 = 0; c0 < h->N; c0 += chunk) {
        const int cnt = std::min(chunk, h->N - c0);
        rc = deliver_output(h, dev + (size_t)c0 * h->cbytes, cnt, dtype, on_device, h->ws + h->cv.stage_a,
                            static_cast<char*>(psi) + (size_t)c0 * eb);
        if (rc) return rc;
        if (!on_device && dtype != h->cfg.compute_dtype) CU(cudaStreamSynchronize(h->stream));
    }
    if (!on_device) CU(cudaStreamSynchronize(h->stream));
    return LBM_OK;
}

int lbm_get_lattice(int lattice, int* q, int* e, double* w, int* opposite_out) {
    if (lattice != LBM_D2Q9 && lattice != LBM_D3Q19) return LBM_E_INVALID;
    auto fill = [&](auto L) {
        using LT = decltype(L);
        if (q) *q = LT::Q;
        for (int i = 0; i < LT::Q; ++i) {
            if (e) for (int a = 0; a < 3; ++a) e[3 * i + a] = LT::E[i][a];
            if (w) w[i] = (double)LT::WN[i] / (double)LT::WD;
            if (opposite_out) opposite_out[i] = opposite<LT>(i);
        }
    };
    if (lattice == LBM_D2Q9) fill(D2Q9{});
    else fill(D3Q19{});
    return LBM_OK;
}

int lbm_halo_bytes(lbm_t* h, int width, size_t* bytes) {
    if (!h || !bytes) return LBM_E_INVALID;
    HaloGeom g;
    const int rc = halo_geom(h, width, &g);
    if (rc) return rc;
    *bytes = (size_t)g.chunk_bytes * (size_t)g.rows;
    return LBM_OK;
}

int lbm_export_halo(lbm_t* h, int side, int width, void* d_buf) {
    if (!h || !d_buf || (side != 0 && side != 1)) return LBM_E_INVALID;
    HaloGeom g;
    int rc = halo_geom(h, width, &g);
    if (rc) return rc;
    if ((rc = halo_ready(h))) return rc;
    return halo_copy(h, g, side == 0 ? width : g.nl - 2LL * width, d_buf, true);
}

int lbm_import_halo(lbm_t* h, int side, int width, const void* d_buf) {
    if (!h || !d_buf || (side != 0 && side != 1)) return LBM_E_INVALID;
    HaloGeom g;
    int rc = halo_geom(h, width, &g);
    if (rc) return rc;
    if ((rc = halo_ready(h))) return rc;
    return halo_copy(h, g, side == 0 ? 0 : g.nl - (long long)width, const_cast<void*>(d_buf), false);
}

size_t lbm_noalloc_max_scratch_bytes(void) { return (size_t)LBM_NOALLOC_SCRATCH_BYTES; }
const char* lbm_noalloc_last_error(void) { return g_noalloc_err.c_str(); }

int lbm_step_noalloc(const lbm_config_t* cfg, const void* d_f_in, void* d_f_out, lbm_stream_t stream) {
    g_noalloc_err.clear();
    int rc = check_config(cfg);
    if (rc != LBM_OK) return noalloc_fail(rc, "lbm_step_noalloc: invalid configuration");
    const lbm_config_t& c = *cfg;
    const int d = c.lattice == LBM_D2Q9 ? 2 : 3;
    for (int a = 0; a < d; ++a)
        if (!c.periodic[a]) return noalloc_fail(LBM_E_UNSUPPORTED, "lbm_step_noalloc: fully periodic domains only (no faces, no solid mask)");
    if (c.flags & LBM_FLAG_NO_COLLIDE) return noalloc_fail(LBM_E_UNSUPPORTED, "lbm_step_noalloc: LBM_FLAG_NO_COLLIDE is not built");
    if (c.zc_A[0] != 0.0 || c.st_kappa[0] != 0.0 || (c.n_components > 1 && (c.zc_A[1] != 0.0 || c.st_kappa[1] != 0.0)))
        return noalloc_fail(LBM_E_UNSUPPORTED, "lbm_step_noalloc: plain Shan-Chen force only (no Zhang-Chen weight, no surface-tension source)");
    const size_t cb = dtype_bytes(c.compute_dtype);
    const size_t N = (size_t)c.nx * c.ny * c.nz;
    const size_t need = (size_t)c.n_components * N * cb;
    if (need > (size_t)LBM_NOALLOC_SCRATCH_BYTES)
        return noalloc_fail(LBM_E_NOMEM, "lbm_step_noalloc: psi of this domain needs " + std::to_string(need) +
                                             " bytes, the static scratch array holds " + std::to_string((size_t)LBM_NOALLOC_SCRATCH_BYTES) +
                                             " (n_components * nx * ny * nz * sizeof(compute dtype) must not exceed it)");
    if (!d_f_in || !d_f_out || d_f_in == d_f_out || ((uintptr_t)d_f_in % cb) != 0 || ((uintptr_t)d_f_out % cb) != 0)
        return noalloc_fail(LBM_E_INVALID, "lbm_step_noalloc: f_in / f_out must be distinct device arrays aligned to the compute dtype");
    void* scratch = nullptr;
    if ((rc = noalloc_scratch(&scratch))) return rc;
    // the kernel parameter block through the same code as the resident path: a handle-shaped record on the host stack
    lbm t = lbm();
    t.cfg = c;
    t.q = q_of(c.lattice);
    t.d = d;
    t.N = (int)N;
    t.plane = (long long)N;
    t.sbytes = cb;
    t.cbytes = cb;
    t.ws = static_cast<char*>(scratch);
    std::memset(&t.cv, 0, sizeof t.cv);
    t.nbsolid = 0;
    t.nfluid = (int)N;
    t.nbr_stride = 0;
    t.snbr_stride = 0;
    t.force_rho = false;
    for (int f = 0; f < 6; ++f) {
        t.face_kind[f] = LBM_FACE_PERIODIC;
        t.face_rho[f][0] = t.face_rho[f][1] = 1.0;
        t.face_u[f][0] = t.face_u[f][1] = t.face_u[f][2] = 0.0;
    }
    cudaError_t e;
    if (c.compute_dtype == LBM_F32) {
        const KParams<float> p = make_params<float>(&t, 0, 0);
        e = noalloc_dispatch<float>(c, p, d_f_in, scratch, d_f_out, static_cast<cudaStream_t>(stream));
    } else {
        const KParams<double> p = make_params<double>(&t, 0, 0);
        e = noalloc_dispatch<double>(c, p, d_f_in, scratch, d_f_out, static_cast<cudaStream_t>(stream));
    }
    if (e != cudaSuccess) return noalloc_fail(LBM_E_CUDA, std::string("lbm_step_noalloc launch: ") + cudaGetErrorString(e));
    return LBM_OK;
}

int lbm_hot_path(const lbm_t* h) { return h ? h->last_path : LBM_E_INVALID; }
int64_t lbm_steps_done(const lbm_t* h) { return h ? h->steps : LBM_E_INVALID; }
int64_t lbm_kernel_launches(const lbm_t* h) { return h ? h->launches : LBM_E_INVALID; }
const char* lbm_last_error(const lbm_t* h) { return h ? h->err.c_str() : "null handle"; }
size_t lbm_config_bytes(void) { return sizeof(lbm_config_t); }
const char* lbm_version(void) { return "paper_2506_17713_b200 0.1 (sm_100a)"; }

}  // extern "C"
