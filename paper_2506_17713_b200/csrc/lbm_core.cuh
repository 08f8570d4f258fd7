// lbm_core.cuh -- device code of the Shan-Chen LBM step for sm_100a.
//
// Kernels (SURVEY.md section 8(a) step numbers; paper citations P:<line> = PAPER.md line):
//   k_moments_v        K1   (lbm_hot.cuh) S1 (rho only) + S3: rho^k = sum_i f_i^k (Eq. 4/10), psi^k (Eq. 12)
//   k_virtual_density  K1b  S2 (+S3 there): improved virtual density at boundary solids (Eq. 17)
//   k_step_v           K2   (lbm_hot.cuh) S1 (j) + S4..S7 fused: pull-stream, force (Eq. 13), common
//                           velocity, BGK/MRT collision (Eq. 3), EDM / shift forcing (Eq. 5),
//                           halfway bounce-back and inlet/outlet faces
//   k_init, k_unstream, k_export_*, k_import_pop   S0 and S8, off the hot loop (this file).
//
// Storage: populations are SoA planes [component][direction][cell], x fastest, in the storage
// dtype ST; arithmetic is in the compute dtype CT.  Between steps the planes hold the POST-COLLISION
// populations f*_i(x,t) with every boundary rule already applied at the writing cell, so that the
// pull of the next step is pure indexing: f_i(x,t+1) = stored_i(x - e_i), or stored_ibar(x) when the
// link flag of direction i is set (source solid / beyond a non-periodic face).  lbm_init_fields /
// lbm_set_populations produce post-stream values f(x,0); k_unstream scatters them once into this
// storage convention (stored_i(x - e_i) = f_i(x), or stored_ibar(x) = f_i(x) on a flagged link), so the
// hot kernels never see a special first step.
#pragma once
#include <cuda_runtime.h>
#include <cuda_fp16.h>
#include <stdint.h>

namespace lbmk {

// ------------------------------------------------------------------ compile-time loop
template <int I> struct IC { static constexpr int value = I; constexpr operator int() const { return I; } };
template <int B, int E, class F>
__host__ __device__ __forceinline__ void static_for(F&& f) {
    if constexpr (B < E) {
        f(IC<B>{});
        static_for<B + 1, E>(static_cast<F&&>(f));
    }
}

// ------------------------------------------------------------------ lattices (R1)
struct D2Q9 {
    static constexpr int D = 2, Q = 9;
    static constexpr int E[9][3] = {{0, 0, 0}, {1, 0, 0}, {-1, 0, 0}, {0, 1, 0}, {0, -1, 0},
                                    {1, 1, 0}, {-1, -1, 0}, {1, -1, 0}, {-1, 1, 0}};
    // weights as rationals: W = WN / 36
    static constexpr int WN[9] = {16, 4, 4, 4, 4, 1, 1, 1, 1};
    static constexpr int WD = 36;
};
struct D3Q19 {
    static constexpr int D = 3, Q = 19;
    static constexpr int E[19][3] = {{0, 0, 0},
                                     {1, 0, 0}, {-1, 0, 0}, {0, 1, 0}, {0, -1, 0}, {0, 0, 1}, {0, 0, -1},
                                     {1, 1, 0}, {-1, -1, 0}, {1, -1, 0}, {-1, 1, 0},
                                     {1, 0, 1}, {-1, 0, -1}, {1, 0, -1}, {-1, 0, 1},
                                     {0, 1, 1}, {0, -1, -1}, {0, 1, -1}, {0, -1, 1}};
    static constexpr int WN[19] = {12, 2, 2, 2, 2, 2, 2, 1, 1, 1, 1, 1, 1, 1, 1, 1, 1, 1, 1};
    static constexpr int WD = 36;
};

template <class L>
constexpr int opposite(int i) {
    for (int k = 0; k < L::Q; ++k)
        if (L::E[k][0] == -L::E[i][0] && L::E[k][1] == -L::E[i][1] && L::E[k][2] == -L::E[i][2]) return k;
    return -1;
}

// MRT moment polynomials (R9, moment order of Eq. 15 P:152 for D2Q9; d'Humieres 2002 for D3Q19).
// Entries are integers; mrt_entry2 returns twice the entry so that the half-integers of row 2 stay integral.
template <class L>
constexpr int mrt_entry2(int r, int i) {
    const int cx = L::E[i][0], cy = L::E[i][1], cz = L::E[i][2];
    const int c2 = cx * cx + cy * cy + cz * cz;
    if (L::D == 2) {
        switch (r) {
            case 0: return 2;
            case 1: return 2 * (-4 + 3 * c2);
            case 2: return 8 - 21 * c2 + 9 * c2 * c2;
            case 3: return 2 * cx;
            case 4: return 2 * (-5 + 3 * c2) * cx;
            case 5: return 2 * cy;
            case 6: return 2 * (-5 + 3 * c2) * cy;
            case 7: return 2 * (cx * cx - cy * cy);
            default: return 2 * cx * cy;
        }
    } else {
        switch (r) {
            case 0: return 2;
            case 1: return 2 * (19 * c2 - 30);
            case 2: return 21 * c2 * c2 - 53 * c2 + 24;
            case 3: return 2 * cx;
            case 4: return 2 * (5 * c2 - 9) * cx;
            case 5: return 2 * cy;
            case 6: return 2 * (5 * c2 - 9) * cy;
            case 7: return 2 * cz;
            case 8: return 2 * (5 * c2 - 9) * cz;
            case 9: return 2 * (3 * cx * cx - c2);
            case 10: return 2 * (3 * c2 - 5) * (3 * cx * cx - c2);
            case 11: return 2 * (cy * cy - cz * cz);
            case 12: return 2 * (3 * c2 - 5) * (cy * cy - cz * cz);
            case 13: return 2 * cx * cy;
            case 14: return 2 * cy * cz;
            case 15: return 2 * cx * cz;
            case 16: return 2 * (cy * cy - cz * cz) * cx;
            case 17: return 2 * (cz * cz - cx * cx) * cy;
            default: return 2 * (cx * cx - cy * cy) * cz;
        }
    }
}
template <class L>
constexpr int mrt_entry(int r, int i) { return mrt_entry2<L>(r, i) / 2; }
template <class L>
constexpr int mrt_norm2(int r) {
    int s = 0;
    for (int i = 0; i < L::Q; ++i) s += mrt_entry<L>(r, i) * mrt_entry<L>(r, i);
    return s;
}

// ------------------------------------------------------------------ kernel parameters
constexpr uint32_t SOLID_BIT = 0x80000000u;  // cell is solid
constexpr uint32_t FACEBC_BIT = 0x40000000u; // fluid cell with >= 1 link across a velocity/pressure face
constexpr uint32_t LINK_MASK = 0x0007fffeu;  // bits 1..18

enum { PSI_CS = 0, PSI_PR = 1, PSI_VDW = 2, PSI_RK = 3, PSI_RKS = 4, PSI_RHO = 5, PSI_EXP = 6, PSI_SC93 = 7 };
enum { FACE_PERIODIC = 0, FACE_WALL = 1, FACE_VELOCITY = 2, FACE_PRESSURE = 3 };

template <class CT>
struct KParams {
    // geometry
    int nx, ny, nz, N;
    int periodic[3];
    long long plane;   // elements between consecutive direction planes (>= N, multiple of 64)
    // buffers
    const void* f_in;  // [NC][Q][plane] storage dtype
    void* f_out;
    CT* psi;           // [NC][N]
    CT* rho;           // [NC][N]
    const uint32_t* flags;  // [N] (only read when BND)
    const int* bsolid; // boundary-solid list
    int nbsolid;
    const uint32_t* bmask;  // per boundary solid: bit i <=> the neighbour at x + e_i is fluid (NULL: test the flags)
    const int* flist;  // fluid-cell list in brick order (lbm_api.cu VisitOrder; list / compact mode of the hot kernels)
    int nfluid;
    // compact mode (lbm_compact.cuh): neighbour table [(Q-1)][nbr_stride] of extended indices; psi in extended order
    const uint32_t* nbr;
    long long nbr_stride;
    long long cplane;   // elements between consecutive direction planes in compact order (= nbr_stride)
    int compact;
    const uint32_t* snbr;   // compact mode: per boundary solid, the fluid-list index of the cell at x_s + e_i or 0xffffffff: [(Q-1)][snbr_stride]
    long long snbr_stride;  // (NULL: K1b gathers the dense rho field through cell coordinates)
    // mode
    int forcing;       // 0 EDM, 1 SHIFT
    int write_rho;     // K1 also writes rho (needed by K1b and the exports)
    // physics
    CT tau[2], inv_tau[2];
    CT G[2][2];
    CT mrt_ce[2][10][10];  // MRT: M^-1 S M restricted to the even subspace (rest + direction pairs), lbm_hot.cuh
    CT mrt_co[2][9][9];    //      ... and to the odd subspace (pair differences)
    CT mrt_c1[2][19], mrt_c2[2][19], mrt_c3[19];   // D3Q19 MRT in moment space: (1 - s_r)/|M_r|^2, s_r/|M_r|^2, 1/|M_r|^2
    CT c_feq_a[2], c_feq_b[2], c_keep[2];  // f* = c_keep f + c_feq_a feq(u_a) + c_feq_b feq(u + du)  (BGK; lbm_hot.cuh)
    CT wref[19];       // w_i * rho_ref
    int psi_kind[2];
    CT eos_a[2], eos_b[2], eos_RT[2], eos_aalpha[2], eos_sqrtT[2], eos_alpha[2], eos_rho0[2], eos_inv_gkk2[2];
    CT wet_phi[2], wet_drho[2], wet_lo[2], wet_hi[2];
    // Zhang-Chen term (Eq. 11-13): zc[k] != 0 <=> A_kk != 0.  The psi field of such a component holds the SIGNED root
    // s = sign(r) sqrt(|r|), r = 2 (alpha p - cs2 rho) / g_kk, so that both psi = max(s, 0) (Eq. 12, clamp R4) and
    // U = alpha p - cs2 rho = (g_kk / 2) s |s| are available to the force without a second field.
    int zc[2];
    CT zcA[2], zc_hg[2];   // A_kk and g_kk / 2
    CT body[3];            // body force per unit mass (R19): F^k += rho^k a, i.e. du^k += a
    int st_on[2];          // surface-tension control (Eq. 14-16): kappa != 0 (D2Q9 MRT)
    CT st_coef[2][4];      // kappa g_kk {1.5 s_e, -1.5 s_eps, -s_nu, -s_nu} (Eq. 15 with R20)
    int face_kind[6];
    CT face_rho[6][2];
    CT face_u[6][3];
};

// Chunked field transfer descriptor of the off-loop kernels (init / import / export): the kernel
// handles cells [c0, c0+cnt); in[s] / out are indexed by (cell - c0).
template <class CT>
struct FieldIO {
    const CT* in[19];
    CT* out;
    long long out_stride;
    int c0, cnt;
};

// Programmatic dependent launch (small, launch-bound domains: lbm_launch.cuh launches the hot kernels with the
// programmatic-serialisation attribute): let the next kernel's CTAs be scheduled right away, then wait until the previous
// kernel has completed and its writes are visible.  Every hot kernel calls this before it touches global memory, so the
// chain stays ordered; without the launch attribute both instructions do nothing.
__device__ __forceinline__ void pdl_begin() {
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");
}

// ------------------------------------------------------------------ storage conversion
template <class CT, class ST> struct Conv;
template <> struct Conv<float, float> {
    static __device__ __forceinline__ float ld(const float* p) { return __ldg(p); }
    static __device__ __forceinline__ void st(float* p, float v) { *p = v; }
};
template <> struct Conv<double, double> {
    static __device__ __forceinline__ double ld(const double* p) { return __ldg(p); }
    static __device__ __forceinline__ void st(double* p, double v) { *p = v; }
};
template <> struct Conv<float, __half> {
    static __device__ __forceinline__ float ld(const __half* p) {
        return __half2float(__ushort_as_half(__ldg(reinterpret_cast<const unsigned short*>(p))));
    }
    static __device__ __forceinline__ void st(__half* p, float v) { *p = __float2half_rn(v); }
};
template <> struct Conv<double, float> {
    static __device__ __forceinline__ double ld(const float* p) { return (double)__ldg(p); }
    static __device__ __forceinline__ void st(float* p, double v) { *p = __double2float_rn(v); }
};

// ------------------------------------------------------------------ cell geometry
struct Cell {
    int id, x, y, z;
    int sxm, sxp, sym, syp, szm, szp;  // scalar-stencil offsets to x-1, x+1, ... (wrap or clamp, R10)
};

template <class L, class CT>
__device__ __forceinline__ Cell make_cell(const KParams<CT>& p, int id) {
    Cell c;
    c.id = id;
    c.x = id % p.nx;
    const int t = id / p.nx;
    c.y = t % p.ny;
    c.z = t / p.ny;
    const int sy = p.nx, sz = p.nx * p.ny;
    c.sxm = c.x > 0 ? -1 : (p.periodic[0] ? p.nx - 1 : 0);
    c.sxp = c.x < p.nx - 1 ? 1 : (p.periodic[0] ? -(p.nx - 1) : 0);
    c.sym = c.y > 0 ? -sy : (p.periodic[1] ? (p.ny - 1) * sy : 0);
    c.syp = c.y < p.ny - 1 ? sy : (p.periodic[1] ? -(p.ny - 1) * sy : 0);
    if constexpr (L::D == 3) {
        c.szm = c.z > 0 ? -sz : (p.periodic[2] ? (p.nz - 1) * sz : 0);
        c.szp = c.z < p.nz - 1 ? sz : (p.periodic[2] ? -(p.nz - 1) * sz : 0);
    } else {
        c.szm = c.szp = 0;
    }
    return c;
}

// offset from the cell to its neighbour at +(ex,ey,ez)
template <int ex, int ey, int ez>
__device__ __forceinline__ int nbr_offset(const Cell& c) {
    int o = 0;
    if constexpr (ex == 1) o += c.sxp;
    if constexpr (ex == -1) o += c.sxm;
    if constexpr (ey == 1) o += c.syp;
    if constexpr (ey == -1) o += c.sym;
    if constexpr (ez == 1) o += c.szp;
    if constexpr (ez == -1) o += c.szm;
    return o;
}

// S7 read side: the Q populations arriving at the cell.
template <class L, class CT, class ST, bool BND>
__device__ __forceinline__ void pull(const KParams<CT>& p, const Cell& c, uint32_t fl, int k, CT (&f)[L::Q]) {
    const ST* base = static_cast<const ST*>(p.f_in) + (long long)k * L::Q * p.plane;
    static_for<0, L::Q>([&](auto I) {
        constexpr int i = I;
        constexpr int ex = L::E[i][0], ey = L::E[i][1], ez = L::E[i][2];
        constexpr int ib = opposite<L>(i);
        const ST* src = base + (long long)i * p.plane + c.id;
        if constexpr (i > 0) {
            int off = nbr_offset<-ex, -ey, -ez>(c);
            if constexpr (BND) {
                if ((fl >> i) & 1u) src = base + (long long)ib * p.plane + c.id;
                else src += off;
            } else {
                src += off;
            }
        }
        f[i] = Conv<CT, ST>::ld(src) + p.wref[i];
    });
}

// ------------------------------------------------------------------ pseudopotential (S3)
// Division and root of the EOS evaluation.  fp32: the hardware approximations (<= 2 ulp) -- the evaluation sits on the
// critical path of the one-pass kernel's producers, and IEEE division / root cost ~10 instructions each; fp64: exact.
__device__ __forceinline__ double eos_div(double a, double b) { return a / b; }
#ifdef LBM_EXACT_EOS
__device__ __forceinline__ float eos_div(float a, float b) { return a / b; }
__device__ __forceinline__ float eos_sqrt(float x) { return sqrtf(x); }
#else
__device__ __forceinline__ float eos_div(float a, float b) { return __fdividef(a, b); }
__device__ __forceinline__ float eos_sqrt(float x) {
    float r;
    asm("sqrt.approx.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
#endif
__device__ __forceinline__ double eos_sqrt(double x) { return sqrt(x); }

template <class CT>
__device__ __forceinline__ CT psi_of_rho(const KParams<CT>& p, int k, CT r) {
    const int kind = p.psi_kind[k];
    if (kind == PSI_RHO) return r;
    if (kind == PSI_EXP) return r > CT(0) ? exp(-CT(1) / r) : CT(0);
    if (kind == PSI_SC93) return p.eos_rho0[k] * (CT(1) - exp(-r / p.eos_rho0[k]));
    const CT a = p.eos_a[k], b = p.eos_b[k], RT = p.eos_RT[k];
    CT pe;
    if (kind == PSI_CS) {
        const CT eta = b * r * CT(0.25);
        const CT om = CT(1) - eta;
        pe = eos_div(r * RT * (CT(1) + eta + eta * eta - eta * eta * eta), om * om * om) - a * r * r;
    } else if (kind == PSI_PR) {
        pe = eos_div(r * RT, CT(1) - b * r) - eos_div(p.eos_aalpha[k] * r * r, CT(1) + CT(2) * b * r - b * b * r * r);
    } else if (kind == PSI_VDW) {
        pe = eos_div(r * RT, CT(1) - b * r) - a * r * r;
    } else if (kind == PSI_RK) {
        pe = eos_div(r * RT, CT(1) - b * r) - eos_div(a * r * r, p.eos_sqrtT[k] * (CT(1) + b * r));
    } else {  // PSI_RKS
        pe = eos_div(r * RT, CT(1) - b * r) - eos_div(p.eos_aalpha[k] * r * r, CT(1) + b * r);
    }
    // Eq. 12: psi = sqrt(2 (alpha p - cs2 rho) / g_kk), radicand clamped at 0 (R4); eos_inv_gkk2 = 2 / g_kk
    const CT rad = (p.eos_alpha[k] * pe - r * CT(1.0 / 3.0)) * p.eos_inv_gkk2[k];
    const CT sq = eos_sqrt(fabs(rad));   // one root; negative radicand: 0 (R4), or the signed root for a Zhang-Chen component
    return rad > CT(0) ? sq : (p.zc[k] ? -sq : CT(0));
}

// f_eq (R1): w_i rho [1 + 3 e.u + 4.5 (e.u)^2 - 1.5 u.u]
template <class L, int i, class CT>
__device__ __forceinline__ CT feq(CT r, const CT (&u)[3], CT uu15) {
    constexpr int ex = L::E[i][0], ey = L::E[i][1], ez = L::E[i][2];
    constexpr CT w = CT(L::WN[i]) / CT(L::WD);
    CT eu = CT(0);
    if constexpr (ex == 1) eu += u[0];
    if constexpr (ex == -1) eu -= u[0];
    if constexpr (ey == 1) eu += u[1];
    if constexpr (ey == -1) eu -= u[1];
    if constexpr (ez == 1) eu += u[2];
    if constexpr (ez == -1) eu -= u[2];
    return w * r * (CT(1) + CT(3) * eu + CT(4.5) * eu * eu - uu15);
}

// ------------------------------------------------------------------ K1b: virtual density at boundary solids
template <class L, int NC, class CT>
__global__ void __launch_bounds__(128) k_virtual_density(const __grid_constant__ KParams<CT> p) {
    pdl_begin();
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= p.nbsolid) return;
    const int id = __ldg(p.bsolid + b);
    const Cell c = make_cell<L>(p, id);
    CT num[NC], den = CT(0);
#pragma unroll
    for (int k = 0; k < NC; ++k) num[k] = CT(0);
    const uint32_t fm = p.bmask ? __ldg(p.bmask + b) : 0u;
    static_for<1, L::Q>([&](auto I) {
        constexpr int i = I;
        constexpr CT w = CT(L::WN[i]) / CT(L::WD);
        const int nb = id + nbr_offset<L::E[i][0], L::E[i][1], L::E[i][2]>(c);
        if (p.bmask ? ((fm >> i) & 1u) != 0u : !(__ldg(p.flags + nb) & SOLID_BIT)) {
            den += w;
#pragma unroll
            for (int k = 0; k < NC; ++k) num[k] += w * p.rho[(long long)k * p.N + nb];
        }
    });
#pragma unroll
    for (int k = 0; k < NC; ++k) {
        CT rs = p.wet_phi[k] * (num[k] / den) - p.wet_drho[k];
        rs = rs < p.wet_lo[k] ? p.wet_lo[k] : rs;
        rs = rs > p.wet_hi[k] ? p.wet_hi[k] : rs;
        p.rho[(long long)k * p.N + id] = rs;
        p.psi[(long long)k * p.N + (p.compact ? p.nfluid + b : id)] = psi_of_rho(p, k, rs);
    }
}

// ------------------------------------------------------------------ shared pieces of K2 / export
// S4: S[kp][a] = sum_i (w_i/cs2) psi^kp(x+e_i) e_ia and, for components with a Zhang-Chen weight,
// Z[kp][a] = sum_i (w_i/cs2) U^kp(x+e_i) e_ia (psi field = signed root there, see KParams::zc)
template <class L, int NC, class CT>
__device__ __forceinline__ void psi_gradient_sums(const KParams<CT>& p, const Cell& c, CT (&S)[NC][3], CT (&Z)[NC][3]) {
#pragma unroll
    for (int kp = 0; kp < NC; ++kp) {
        S[kp][0] = S[kp][1] = S[kp][2] = CT(0);
        Z[kp][0] = Z[kp][1] = Z[kp][2] = CT(0);
        const CT* ps = p.psi + (long long)kp * p.N + c.id;
        const bool zc = p.zc[kp] != 0;
        static_for<1, L::Q>([&](auto I) {
            constexpr int i = I;
            constexpr int ex = L::E[i][0], ey = L::E[i][1], ez = L::E[i][2];
            constexpr CT gw = CT(3 * L::WN[i]) / CT(L::WD);
            const CT s = __ldg(ps + nbr_offset<ex, ey, ez>(c));
            const CT v = gw * (zc && s < CT(0) ? CT(0) : s);
            if constexpr (ex == 1) S[kp][0] += v;
            if constexpr (ex == -1) S[kp][0] -= v;
            if constexpr (ey == 1) S[kp][1] += v;
            if constexpr (ey == -1) S[kp][1] -= v;
            if constexpr (ez == 1) S[kp][2] += v;
            if constexpr (ez == -1) S[kp][2] -= v;
            if (zc) {
                const CT u = gw * (p.zc_hg[kp] * s * fabs(s));
                if constexpr (ex == 1) Z[kp][0] += u;
                if constexpr (ex == -1) Z[kp][0] -= u;
                if constexpr (ey == 1) Z[kp][1] += u;
                if constexpr (ey == -1) Z[kp][1] -= u;
                if constexpr (ez == 1) Z[kp][2] += u;
                if constexpr (ez == -1) Z[kp][2] -= u;
            }
        });
    }
}

// which non-periodic face does the link from the cell along +e_o cross (lowest axis first)? -1 = none
template <class L, int o, class CT>
__device__ __forceinline__ int crossed_face(const KParams<CT>& p, const Cell& c) {
    constexpr int ex = L::E[o][0], ey = L::E[o][1], ez = L::E[o][2];
    if constexpr (ex != 0) {
        if (!p.periodic[0]) {
            if (ex < 0 && c.x == 0) return 0;
            if (ex > 0 && c.x == p.nx - 1) return 1;
        }
    }
    if constexpr (ey != 0) {
        if (!p.periodic[1]) {
            if (ey < 0 && c.y == 0) return 2;
            if (ey > 0 && c.y == p.ny - 1) return 3;
        }
    }
    if constexpr (ez != 0 && L::D == 3) {
        if (!p.periodic[2]) {
            if (ez < 0 && c.z == 0) return 4;
            if (ez > 0 && c.z == p.nz - 1) return 5;
        }
    }
    return -1;
}

// ------------------------------------------------------------------ S0: initialisation
// io.in[k] = rho^k, io.in[2+a] = u_a (NULL = 0) for cells [c0, c0+cnt)
template <class L, int NC, class CT, class ST>
__global__ void __launch_bounds__(256) k_init(const __grid_constant__ KParams<CT> p, const __grid_constant__ FieldIO<CT> io,
                                             void* f_other, int has_flags) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= io.cnt) return;
    const int id = io.c0 + t;
    const bool solid = has_flags && (__ldg(p.flags + id) & SOLID_BIT);
#pragma unroll
    for (int k = 0; k < NC; ++k) {
        CT r = CT(1);
        CT u[3] = {CT(0), CT(0), CT(0)};
        if (!solid) {
            r = io.in[k][t];
#pragma unroll
            for (int a = 0; a < L::D; ++a)
                if (io.in[2 + a]) u[a] = io.in[2 + a][t];
        }
        const CT uu15 = CT(1.5) * (u[0] * u[0] + u[1] * u[1] + u[2] * u[2]);
        ST* a_ = static_cast<ST*>(p.f_out) + (long long)k * L::Q * p.plane + id;
        ST* b_ = static_cast<ST*>(f_other) + (long long)k * L::Q * p.plane + id;
        static_for<0, L::Q>([&](auto I) {
            constexpr int i = I;
            const CT v = feq<L, i, CT>(r, u, uu15) - p.wref[i];
            Conv<CT, ST>::st(a_ + (long long)i * p.plane, v);
            Conv<CT, ST>::st(b_ + (long long)i * p.plane, v);
        });
    }
}

// Post-stream f(x,0) in f_in  ->  storage convention in f_out (see the header of this file): a pure scatter of
// stored values (no arithmetic), race-free because every slot has at most one writer; slots nobody writes keep
// the copy k_init / k_import_pop left there.
template <class L, int NC, class ST, class CT, bool BND>
__global__ void __launch_bounds__(256) k_unstream(const __grid_constant__ KParams<CT> p, int only_k /* -1 = all */) {
    const int id = blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= p.N) return;
    uint32_t fl = 0;
    if constexpr (BND) {
        fl = __ldg(p.flags + id);
        if (fl & SOLID_BIT) return;
    }
    const Cell c = make_cell<L>(p, id);
#pragma unroll
    for (int k = 0; k < NC; ++k) {
        if (only_k >= 0 && k != only_k) continue;
        const ST* in = static_cast<const ST*>(p.f_in) + (long long)k * L::Q * p.plane + id;
        ST* out = static_cast<ST*>(p.f_out) + (long long)k * L::Q * p.plane + id;
        static_for<0, L::Q>([&](auto I) {
            constexpr int i = I;
            constexpr int ib = opposite<L>(i);
            const ST v = in[(long long)i * p.plane];
            if constexpr (i == 0) {
                out[0] = v;
            } else {
                if (BND && ((fl >> i) & 1u)) out[(long long)ib * p.plane] = v;
                else out[(long long)i * p.plane + nbr_offset<-L::E[i][0], -L::E[i][1], -L::E[i][2]>(c)] = v;
            }
        });
    }
}

// ------------------------------------------------------------------ S8: exports
// rho (from the rho field refreshed by K1/K1b), u = (sum j + F/2)/sum rho, p = cs2 sum rho + 1/2 sum g psi psi'
template <class L, int NC, class CT, class ST, bool BND>
__global__ void __launch_bounds__(128) k_export_macro(const __grid_constant__ KParams<CT> p, CT* __restrict__ u_out,
                                                     CT* __restrict__ p_out) {
    const int id = blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= p.N) return;
    uint32_t fl = 0;
    if constexpr (BND) fl = __ldg(p.flags + id);
    if (fl & SOLID_BIT) {
        if (u_out)
            for (int a = 0; a < L::D; ++a) u_out[(long long)a * p.N + id] = CT(0);
        if (p_out) p_out[id] = CT(0);
        return;
    }
    const Cell c = make_cell<L>(p, id);
    CT rho[NC], j[NC][3];
#pragma unroll
    for (int k = 0; k < NC; ++k) {
        CT f[L::Q];
        pull<L, CT, ST, BND>(p, c, fl, k, f);
        CT r = CT(0), jx = CT(0), jy = CT(0), jz = CT(0);
        static_for<0, L::Q>([&](auto I) {
            constexpr int i = I;
            const CT v = f[i];
            r += v;
            if constexpr (L::E[i][0] == 1) jx += v;
            if constexpr (L::E[i][0] == -1) jx -= v;
            if constexpr (L::E[i][1] == 1) jy += v;
            if constexpr (L::E[i][1] == -1) jy -= v;
            if constexpr (L::E[i][2] == 1) jz += v;
            if constexpr (L::E[i][2] == -1) jz -= v;
        });
        rho[k] = r; j[k][0] = jx; j[k][1] = jy; j[k][2] = jz;
    }
    CT S[NC][3], Z[NC][3];
    psi_gradient_sums<L, NC, CT>(p, c, S, Z);
    CT psi[NC], rt = CT(0);
#pragma unroll
    for (int k = 0; k < NC; ++k) {
        psi[k] = p.psi[(long long)k * p.N + id];
        if (p.zc[k] && psi[k] < CT(0)) psi[k] = CT(0);
        rt += rho[k];
    }
    if (u_out) {
#pragma unroll
        for (int a = 0; a < L::D; ++a) {
            CT js = CT(0), Fs = CT(0);
#pragma unroll
            for (int k = 0; k < NC; ++k) {
                CT acc = CT(0);
#pragma unroll
                for (int kp = 0; kp < NC; ++kp) acc += p.G[k][kp] * S[kp][a];
                js += j[k][a];
                Fs += p.zc[k] ? (CT(1) - p.zcA[k]) * (-psi[k] * acc) - p.zcA[k] * Z[k][a] : -psi[k] * acc;
                Fs += rho[k] * p.body[a];
            }
            u_out[(long long)a * p.N + id] = (js + Fs * CT(0.5)) / rt;
        }
    }
    if (p_out) {
        CT pp = CT(0);
#pragma unroll
        for (int k = 0; k < NC; ++k)
#pragma unroll
            for (int kp = 0; kp < NC; ++kp) pp += p.G[k][kp] * psi[k] * psi[kp];
        p_out[id] = rt * CT(1.0 / 3.0) + pp * CT(0.5);
    }
}

// canonical post-stream populations of one component -> io.out[i*out_stride + (cell - c0)] (compute dtype)
template <class L, class CT, class ST, bool BND>
__global__ void __launch_bounds__(256) k_export_pop(const __grid_constant__ KParams<CT> p, int k,
                                                   const __grid_constant__ FieldIO<CT> io) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= io.cnt) return;
    const int id = io.c0 + t;
    uint32_t fl = 0;
    if constexpr (BND) fl = __ldg(p.flags + id);
    CT f[L::Q];
    if (fl & SOLID_BIT) {
        const ST* base = static_cast<const ST*>(p.f_in) + (long long)k * L::Q * p.plane + id;
        static_for<0, L::Q>([&](auto I) { f[I] = Conv<CT, ST>::ld(base + (long long)I * p.plane) + p.wref[I]; });
    } else {
        const Cell c = make_cell<L>(p, id);
        pull<L, CT, ST, BND>(p, c, fl, k, f);
    }
    static_for<0, L::Q>([&](auto I) { io.out[(long long)I * io.out_stride + t] = f[I]; });
}

// io.in[i][cell - c0] (compute dtype) -> planes of component k in both buffers
template <class L, class CT, class ST>
__global__ void __launch_bounds__(256) k_import_pop(const __grid_constant__ KParams<CT> p, int k,
                                                   const __grid_constant__ FieldIO<CT> io, void* f_other) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= io.cnt) return;
    const int id = io.c0 + t;
    ST* a_ = static_cast<ST*>(p.f_out) + (long long)k * L::Q * p.plane + id;
    ST* b_ = static_cast<ST*>(f_other) + (long long)k * L::Q * p.plane + id;
    static_for<0, L::Q>([&](auto I) {
        const CT v = io.in[I][t] - p.wref[I];
        Conv<CT, ST>::st(a_ + (long long)I * p.plane, v);
        Conv<CT, ST>::st(b_ + (long long)I * p.plane, v);
    });
}

}  // namespace lbmk
