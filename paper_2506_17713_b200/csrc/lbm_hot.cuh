// lbm_hot.cuh -- the hot-loop kernels of the Shan-Chen LBM step for sm_100a.
//
//   k_moments_v  K1   S1 (rho) + S3 (psi)                      Eq. 4/10, Eq. 12
//   k_step_v     K2   S1 (j) + S4..S7 fused                     Eq. 13, Eq. 3, Eq. 5,
//                                                               Eq. 2, bounce-back P:219, faces P:313
//
// Design for B200 (the step is an HBM-bound stencil; the first one-thread-per-cell version was issue-bound at
// ~930 instructions per cell, profiles/r01_*):
//   * every thread owns VEC consecutive cells of one x-row; the population planes are read and written with
//     128-bit (or 64-bit) vector accesses.  Stores are always aligned because the planes hold post-collision
//     values at the cell that computed them; a pull along +-x is the aligned vector of the row plus ONE scalar
//     from the neighbouring vector (an L1 hit);
//   * index arithmetic (two integer divisions, wrap/clamp of the 3x3 row neighbourhood) is paid once per thread;
//   * the arithmetic is organised over the (i, ibar) direction pairs: sums and differences give the moments,
//     the two equilibria of a pair share their even part, and MRT is applied as two small dense blocks
//     (even / odd subspace of M^-1 S M, precomputed on the host) instead of two 19x19 products.
// Summation order therefore differs from the oracle's index order: parity holds to rounding.
#pragma once
#include "lbm_core.cuh"

namespace lbmk {

// ------------------------------------------------------------------ vector load / store in the storage dtype
template <int BYTES> struct RawVec;
template <> struct RawVec<2> { using type = unsigned short; };
template <> struct RawVec<4> { using type = unsigned int; };
template <> struct RawVec<8> { using type = uint2; };
template <> struct RawVec<16> { using type = uint4; };

template <class CT, class ST> struct Cvt;
template <> struct Cvt<float, float> {
    static __device__ __forceinline__ float up(float v) { return v; }
    static __device__ __forceinline__ float down(float v) { return v; }
};
template <> struct Cvt<double, double> {
    static __device__ __forceinline__ double up(double v) { return v; }
    static __device__ __forceinline__ double down(double v) { return v; }
};
template <> struct Cvt<float, __half> {
    static __device__ __forceinline__ float up(__half v) { return __half2float(v); }
    static __device__ __forceinline__ __half down(float v) { return __float2half_rn(v); }  // R16: RNE once, at the store
};
template <> struct Cvt<double, float> {
    static __device__ __forceinline__ double up(float v) { return (double)v; }
    static __device__ __forceinline__ float down(double v) { return __double2float_rn(v); }
};

template <> struct Cvt<uint32_t, uint32_t> {
    static __device__ __forceinline__ uint32_t up(uint32_t v) { return v; }
    static __device__ __forceinline__ uint32_t down(uint32_t v) { return v; }
};

template <class CT, class ST, int VEC>
__device__ __forceinline__ void ld_vec(const ST* __restrict__ p, CT (&out)[VEC]) {
    using R = typename RawVec<sizeof(ST) * VEC>::type;
    const R r = __ldg(reinterpret_cast<const R*>(p));
    const ST* t = reinterpret_cast<const ST*>(&r);
#pragma unroll
    for (int v = 0; v < VEC; ++v) out[v] = Cvt<CT, ST>::up(t[v]);
}
template <class CT, class ST>
__device__ __forceinline__ CT ld_one(const ST* __restrict__ p) {
    CT t[1];
    ld_vec<CT, ST, 1>(p, t);
    return t[0];
}
template <class CT, class ST, int VEC>
__device__ __forceinline__ void st_vec(ST* __restrict__ p, const CT (&in)[VEC]) {
    using R = typename RawVec<sizeof(ST) * VEC>::type;
    R r;
    ST* t = reinterpret_cast<ST*>(&r);
#pragma unroll
    for (int v = 0; v < VEC; ++v) t[v] = Cvt<CT, ST>::down(in[v]);
    *reinterpret_cast<R*>(p) = r;
}

// same, through an explicit st.global (for addresses whose provenance the compiler cannot see: generic ST otherwise)
template <class CT, class ST, int VEC>
__device__ __forceinline__ void st_vec_global(ST* p, const CT (&in)[VEC]) {
    using R = typename RawVec<sizeof(ST) * VEC>::type;
    R r;
    ST* t = reinterpret_cast<ST*>(&r);
#pragma unroll
    for (int v = 0; v < VEC; ++v) t[v] = Cvt<CT, ST>::down(in[v]);
    if constexpr (sizeof(R) == 16) {
        const uint4 u = *reinterpret_cast<const uint4*>(&r);
        asm volatile("st.global.v4.b32 [%0], {%1, %2, %3, %4};" ::"l"(p), "r"(u.x), "r"(u.y), "r"(u.z), "r"(u.w) : "memory");
    } else if constexpr (sizeof(R) == 8) {
        const uint2 u = *reinterpret_cast<const uint2*>(&r);
        asm volatile("st.global.v2.b32 [%0], {%1, %2};" ::"l"(p), "r"(u.x), "r"(u.y) : "memory");
    } else {
        *reinterpret_cast<R*>(p) = r;
    }
}

// ------------------------------------------------------------------ geometry of a thread's VEC cells
struct VCell {
    int id0;       // cell index of lane 0
    int x0, y, z;
    int xm, xp;    // x index left of lane 0 / right of lane VEC-1 (wrap, or clamp on a non-periodic axis: R10)
    int yo[3];     // element offset of rows y-1, y, y+1 (wrap / clamp)
    int zo[3];     // element offset of planes z-1, z, z+1
};

template <class L, int VEC, class CT>
__device__ __forceinline__ VCell make_vcell(const KParams<CT>& p, unsigned vid) {
    VCell c;
    const unsigned nxv = (unsigned)p.nx / VEC;
    const unsigned r = vid / nxv;
    c.x0 = (int)(vid - r * nxv) * VEC;
    if constexpr (L::D == 3) {
        c.z = (int)(r / (unsigned)p.ny);
        c.y = (int)(r - (unsigned)c.z * (unsigned)p.ny);
    } else {
        c.z = 0;
        c.y = (int)r;
    }
    const int sy = p.nx, sz = p.nx * p.ny;
    c.xm = c.x0 > 0 ? c.x0 - 1 : (p.periodic[0] ? p.nx - 1 : 0);
    c.xp = c.x0 + VEC < p.nx ? c.x0 + VEC : (p.periodic[0] ? 0 : p.nx - 1);
    c.yo[1] = c.y * sy;
    c.yo[0] = c.y > 0 ? c.yo[1] - sy : (p.periodic[1] ? (p.ny - 1) * sy : c.yo[1]);
    c.yo[2] = c.y < p.ny - 1 ? c.yo[1] + sy : (p.periodic[1] ? 0 : c.yo[1]);
    if constexpr (L::D == 3) {
        c.zo[1] = c.z * sz;
        c.zo[0] = c.z > 0 ? c.zo[1] - sz : (p.periodic[2] ? (p.nz - 1) * sz : c.zo[1]);
        c.zo[2] = c.z < p.nz - 1 ? c.zo[1] + sz : (p.periodic[2] ? 0 : c.zo[1]);
    } else {
        c.zo[0] = c.zo[1] = c.zo[2] = 0;
    }
    c.id0 = c.zo[1] + c.yo[1] + c.x0;
    return c;
}

// S7 read side for VEC cells: f[i][v] = stored_i(x_v - e_i), or stored_ibar(x_v) on a flagged link.
template <class L, class CT, class ST, bool BND, int VEC>
__device__ __forceinline__ void pull_vec(const KParams<CT>& p, const VCell& c, const uint32_t (&fl)[VEC], int k,
                                         CT (&f)[L::Q][VEC]) {
    const ST* base = static_cast<const ST*>(p.f_in) + (long long)k * L::Q * p.plane;
    uint32_t any = 0;
    if constexpr (BND) {
#pragma unroll
        for (int v = 0; v < VEC; ++v) any |= fl[v];
    }
    static_for<0, L::Q>([&](auto I) {
        constexpr int i = I;
        constexpr int ex = L::E[i][0], ey = L::E[i][1], ez = L::E[i][2];
        const ST* row = base + (long long)i * p.plane + (c.zo[1 - ez] + c.yo[1 - ey]);
        if constexpr (ex == 0) {
            ld_vec<CT, ST, VEC>(row + c.x0, f[i]);
        } else if constexpr (VEC == 1) {
            f[i][0] = ld_one<CT, ST>(row + (ex > 0 ? c.xm : c.xp));
        } else {
            CT t[VEC];
            ld_vec<CT, ST, VEC>(row + c.x0, t);
            if constexpr (ex > 0) {
                f[i][0] = ld_one<CT, ST>(row + c.xm);
#pragma unroll
                for (int v = 1; v < VEC; ++v) f[i][v] = t[v - 1];
            } else {
#pragma unroll
                for (int v = 0; v < VEC - 1; ++v) f[i][v] = t[v + 1];
                f[i][VEC - 1] = ld_one<CT, ST>(row + c.xp);
            }
        }
        if constexpr (BND && i > 0) {
            if ((any >> i) & 1u) {
                constexpr int ib = opposite<L>(i);
                CT own[VEC];
                ld_vec<CT, ST, VEC>(base + (long long)ib * p.plane + c.id0, own);
#pragma unroll
                for (int v = 0; v < VEC; ++v)
                    if ((fl[v] >> i) & 1u) f[i][v] = own[v];
            }
        }
#pragma unroll
        for (int v = 0; v < VEC; ++v) f[i][v] += p.wref[i];
    });
}

// link flags of the thread's cells; returns false when every lane is solid (nothing to do)
template <bool BND, int VEC, class CT>
__device__ __forceinline__ bool load_flags(const KParams<CT>& p, const VCell& c, uint32_t (&fl)[VEC]) {
    if constexpr (!BND) {
#pragma unroll
        for (int v = 0; v < VEC; ++v) fl[v] = 0;
        return true;
    } else {
        ld_vec<uint32_t, uint32_t, VEC>(p.flags + c.id0, fl);
        uint32_t all = SOLID_BIT;
#pragma unroll
        for (int v = 0; v < VEC; ++v) all &= fl[v];
        return all == 0;
    }
}

// store VEC values of one field; solid lanes are skipped
template <class CT, class ST, bool BND, int VEC>
__device__ __forceinline__ void store_lanes(ST* __restrict__ dst, const CT (&val)[VEC], const uint32_t (&fl)[VEC]) {
    if constexpr (BND) {
        uint32_t anys = 0;
#pragma unroll
        for (int v = 0; v < VEC; ++v) anys |= fl[v];
        if (anys & SOLID_BIT) {
#pragma unroll
            for (int v = 0; v < VEC; ++v)
                if (!(fl[v] & SOLID_BIT)) dst[v] = Cvt<CT, ST>::down(val[v]);
            return;
        }
    }
    st_vec<CT, ST, VEC>(dst, val);
}

// ------------------------------------------------------------------ arithmetic over direction pairs
// Both lattices list direction 2p+1 and its opposite 2p+2 next to each other (include/lbm.h).
template <class L>
constexpr bool pairs_ok() {
    for (int pq = 0; pq < (L::Q - 1) / 2; ++pq)
        if (opposite<L>(2 * pq + 1) != 2 * pq + 2) return false;
    return true;
}
static_assert(pairs_ok<D2Q9>() && pairs_ok<D3Q19>(), "direction order must list opposite pairs");

// S1: rho = sum f, j = sum f e  (Eq. 4, 10)
template <class L, class CT>
__device__ __forceinline__ void moments(const CT (&f)[L::Q], CT& rho, CT (&j)[3]) {
    CT r = f[0], jx = CT(0), jy = CT(0), jz = CT(0);
    static_for<0, (L::Q - 1) / 2>([&](auto P) {
        constexpr int a = 2 * P + 1, b = a + 1;
        const CT s = f[a] + f[b], d = f[a] - f[b];
        r += s;
        if constexpr (L::E[a][0] == 1) jx += d;
        if constexpr (L::E[a][0] == -1) jx -= d;
        if constexpr (L::E[a][1] == 1) jy += d;
        if constexpr (L::E[a][1] == -1) jy -= d;
        if constexpr (L::E[a][2] == 1) jz += d;
        if constexpr (L::E[a][2] == -1) jz -= d;
    });
    rho = r; j[0] = jx; j[1] = jy; j[2] = jz;
}
template <class L, class CT>
__device__ __forceinline__ CT density(const CT (&f)[L::Q]) {
    CT r = f[0];
    static_for<0, (L::Q - 1) / 2>([&](auto P) { r += f[2 * P + 1] + f[2 * P + 2]; });
    return r;
}

// acc_i (+)= coef * f_eq,i(rho, u)   (R1: f_eq = w rho [1 + 3 e.u + 4.5 (e.u)^2 - 1.5 u.u]); a pair shares its even part.
// SET: acc_i = ... (the accumulator is not read)
template <class L, class CT, bool SET = false>
__device__ __forceinline__ void add_feq(CT coef, CT rho, const CT (&u)[3], CT (&acc)[L::Q]) {
    const CT cr = coef * rho;
    const CT c0 = CT(1) - CT(1.5) * (u[0] * u[0] + u[1] * u[1] + u[2] * u[2]);
    if constexpr (SET) acc[0] = (cr * (CT(L::WN[0]) / CT(L::WD))) * c0;
    else acc[0] += (cr * (CT(L::WN[0]) / CT(L::WD))) * c0;
    static_for<0, (L::Q - 1) / 2>([&](auto P) {
        constexpr int a = 2 * P + 1, b = a + 1;
        constexpr int ex = L::E[a][0], ey = L::E[a][1], ez = L::E[a][2];
        CT eu = CT(0);
        if constexpr (ex == 1) eu += u[0];
        if constexpr (ex == -1) eu -= u[0];
        if constexpr (ey == 1) eu += u[1];
        if constexpr (ey == -1) eu -= u[1];
        if constexpr (ez == 1) eu += u[2];
        if constexpr (ez == -1) eu -= u[2];
        const CT wr = cr * (CT(L::WN[a]) / CT(L::WD));
        const CT even = c0 + CT(4.5) * eu * eu;
        const CT odd = CT(3) * eu;
        if constexpr (SET) {
            acc[a] = wr * (even + odd);
            acc[b] = wr * (even - odd);
        } else {
            acc[a] += wr * (even + odd);
            acc[b] += wr * (even - odd);
        }
    });
}

// D3Q19 equilibrium moments m_eq = M f_eq(rho, u) in closed form (R9: d'Humieres basis, f_eq of R1; the same expressions
// are held to the oracle's matrix product in tests/test_oracle_basics.py::test_d3q19_equilibrium_moments_closed_form, the
// kernel to the oracle's dense M^-1 S M by the fp64 parity tests): row order of mrt_entry2<D3Q19>.
template <class CT>
__device__ __forceinline__ void meq_d3q19(CT rho, const CT (&u)[3], CT (&m)[19]) {
    const CT jx = rho * u[0], jy = rho * u[1], jz = rho * u[2];
    const CT xx = jx * u[0], yy = jy * u[1], zz = jz * u[2];
    const CT ruu = xx + yy + zz;
    m[0] = rho;
    m[1] = CT(19) * ruu - CT(11) * rho;
    m[2] = CT(3) * rho - CT(5.5) * ruu;
    m[3] = jx; m[4] = CT(-2.0 / 3.0) * jx;
    m[5] = jy; m[6] = CT(-2.0 / 3.0) * jy;
    m[7] = jz; m[8] = CT(-2.0 / 3.0) * jz;
    m[9] = CT(2) * xx - yy - zz;
    m[10] = CT(-0.5) * m[9];
    m[11] = yy - zz;
    m[12] = CT(-0.5) * m[11];
    m[13] = jx * u[1];
    m[14] = jy * u[2];
    m[15] = jx * u[2];
    m[16] = m[17] = m[18] = CT(0);
}

// S6, MRT on D3Q19 in moment space (Eq. 3 second line):  f* = M^-1 [ m - S (m - m_eq(u_a)) (+ m_eq(u_b) - m_eq(u') for
// EDM, Eq. 5) ].  The rows of M are even or odd polynomials of c, so the transform splits into the pair sums (10 even
// moments) and the pair differences (9 odd moments); its integer entries (0, +-1, +-2, +-4, 8, -11, 12, -30) are factored by
// hand: ~50 additions forward, ~90 multiply-adds back, instead of the 181 multiply-adds of the dense even / odd blocks plus
// a second 19-term f_eq.  c1 = (1 - s_r) / |M_r|^2, c2 = s_r / |M_r|^2, c3 = 1 / |M_r|^2 come from the host.
template <class CT>
__device__ __forceinline__ void collide_mrt_d3q19(const KParams<CT>& p, int k, CT rho, const CT (&u)[3], const CT (&ua)[3],
                                                  const CT (&ub)[3], bool edm, CT (&f)[19]) {
    (void)u;   // EDM: u_a = u'
    // pair sums / differences: x, y, z, xy+, xy-, xz+, xz-, yz+, yz-  (directions 2P+1, 2P+2)
    const CT sx = f[1] + f[2], sy = f[3] + f[4], sz = f[5] + f[6];
    const CT sa = f[7] + f[8], sb = f[9] + f[10], sc = f[11] + f[12], sd = f[13] + f[14], sg = f[15] + f[16], sh = f[17] + f[18];
    const CT dx = f[1] - f[2], dy = f[3] - f[4], dz = f[5] - f[6];
    const CT da = f[7] - f[8], db = f[9] - f[10], dc = f[11] - f[12], dd = f[13] - f[14], dg = f[15] - f[16], dh = f[17] - f[18];
    CT m[19];
    {   // even moments
        const CT A = sx + sy + sz, Sxy = sa + sb, Sxz = sc + sd, Syz = sg + sh, D = Sxy + Sxz + Syz;
        const CT t9 = Sxy + Sxz - CT(2) * Syz, t11 = Sxy - Sxz;
        const CT ax = CT(2) * sx - sy - sz, aw = sy - sz;
        m[0] = f[0] + A + D;
        m[1] = CT(8) * D - CT(11) * A - CT(30) * f[0];
        m[2] = D - CT(4) * A + CT(12) * f[0];
        m[9] = ax + t9;
        m[10] = t9 - CT(2) * ax;
        m[11] = aw + t11;
        m[12] = t11 - CT(2) * aw;
        m[13] = sa - sb;
        m[14] = sg - sh;
        m[15] = sc - sd;
    }
    {   // odd moments
        const CT ox = da + db + dc + dd, oy = da - db + dg + dh, oz = dc - dd + dg - dh;
        m[3] = dx + ox; m[4] = ox - CT(4) * dx;
        m[5] = dy + oy; m[6] = oy - CT(4) * dy;
        m[7] = dz + oz; m[8] = oz - CT(4) * dz;
        m[16] = da + db - dc - dd;
        m[17] = db - da + dg + dh;
        m[18] = dc - dd - dg + dh;
    }
    // relaxation towards m_eq(u_a), EDM source m_eq(u_b) - m_eq(u'); the result is already divided by |M_r|^2
    CT me[19];
    meq_d3q19<CT>(rho, ua, me);
    static_for<0, 19>([&](auto R) { m[R] = p.mrt_c1[k][R] * m[R] + p.mrt_c2[k][R] * me[R]; });
    if (edm) {
        CT mb[19];
        meq_d3q19<CT>(rho, ub, mb);
        static_for<1, 16>([&](auto R) { m[R] += p.mrt_c3[R] * (mb[R] - me[R]); });
    }
    // back: f = M^T m
    {
        const CT base_a = m[0] - CT(11) * m[1] - CT(4) * m[2];      // axis directions
        const CT base_d = m[0] + CT(8) * m[1] + m[2];               // diagonals
        const CT q9 = m[9] + m[10], q11 = m[11] + m[12];
        const CT ex_ = base_a + CT(2) * m[9] - CT(4) * m[10];
        const CT ey_ = base_a - m[9] + CT(2) * m[10] + m[11] - CT(2) * m[12];
        const CT ez_ = base_a - m[9] + CT(2) * m[10] - m[11] + CT(2) * m[12];
        const CT exy = base_d + q9 + q11, exz = base_d + q9 - q11, eyz = base_d - CT(2) * q9;
        const CT ox_ = m[3] - CT(4) * m[4], oy_ = m[5] - CT(4) * m[6], oz_ = m[7] - CT(4) * m[8];
        const CT jqx = m[3] + m[4], jqy = m[5] + m[6], jqz = m[7] + m[8];
        f[0] = m[0] - CT(30) * m[1] + CT(12) * m[2];
        f[1] = ex_ + ox_; f[2] = ex_ - ox_;
        f[3] = ey_ + oy_; f[4] = ey_ - oy_;
        f[5] = ez_ + oz_; f[6] = ez_ - oz_;
        {   // (1,1,0) / (1,-1,0)
            const CT ea = exy + m[13], eb = exy - m[13];
            const CT oa = jqx + jqy + m[16] - m[17], ob = jqx - jqy + m[16] + m[17];
            f[7] = ea + oa; f[8] = ea - oa; f[9] = eb + ob; f[10] = eb - ob;
        }
        {   // (1,0,1) / (1,0,-1)
            const CT ea = exz + m[15], eb = exz - m[15];
            const CT oa = jqx + jqz - m[16] + m[18], ob = jqx - jqz - m[16] - m[18];
            f[11] = ea + oa; f[12] = ea - oa; f[13] = eb + ob; f[14] = eb - ob;
        }
        {   // (0,1,1) / (0,1,-1)
            const CT ea = eyz + m[14], eb = eyz - m[14];
            const CT oa = jqy + jqz + m[17] - m[18], ob = jqy - jqz + m[17] + m[18];
            f[15] = ea + oa; f[16] = ea - oa; f[17] = eb + ob; f[18] = eb - ob;
        }
    }
}

// S6 for one cell and one component.  u: common velocity u' (R6); du = F/rho (Eq. 5).
//   BGK : f* = c_keep f + c_feq_a f_eq(u_a) + c_feq_b f_eq(u' + du)
//         EDM   (Eq. 3 + Eq. 5): u_a = u', c_keep = 1 - 1/tau, c_feq_a = 1/tau - 1, c_feq_b = 1
//         SHIFT (R7)           : u_a = u' + tau du, c_keep = 1 - 1/tau, c_feq_a = 1/tau, c_feq_b = 0
//   MRT : f* = f - M^-1 S M (f - f_eq(u_a)) [+ f_eq(u' + du) - f_eq(u') for EDM].  D3Q19: in moment space with the
//         hand-factored transform (collide_mrt_d3q19).  D2Q9: M^-1 S M applied as its even block (on f_0 and the pair
//         sums) and odd block (on the pair differences): rows of M are even or odd polynomials of c (R9), so
//         M^-1 S M = C_even + C_odd with no cross terms.
template <class L, int COLL, class CT>
__device__ __forceinline__ void collide(const KParams<CT>& p, int k, CT rho, const CT (&u)[3], const CT (&du)[3],
                                        CT (&f)[L::Q]) {
    constexpr int NP = (L::Q - 1) / 2;
    const bool shift = p.forcing == 1;
    CT ua[3], ub[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        ub[a] = u[a] + du[a];
        ua[a] = shift ? u[a] + p.tau[k] * du[a] : u[a];
    }
    if constexpr (COLL == 0) {
        const CT keep = p.c_keep[k], ca = p.c_feq_a[k], cb = p.c_feq_b[k];
        if (keep == CT(0) && ca == CT(0)) {          // tau = 1, EDM: f* = f_eq(rho, u' + du)
            add_feq<L, CT, true>(cb, rho, ub, f);
        } else if (keep == CT(0) && cb == CT(0)) {   // tau = 1, SHIFT: f* = f_eq(rho, u' + tau du)
            add_feq<L, CT, true>(ca, rho, ua, f);
        } else {
            static_for<0, L::Q>([&](auto I) { f[I] *= keep; });
            if (ca != CT(0)) add_feq<L, CT>(ca, rho, ua, f);
            if (cb != CT(0)) add_feq<L, CT>(cb, rho, ub, f);
        }
    } else if constexpr (L::D == 3) {
        collide_mrt_d3q19<CT>(p, k, rho, u, ua, ub, !shift, f);
    } else {
        CT e[L::Q];
        static_for<0, L::Q>([&](auto I) { e[I] = CT(0); });
        add_feq<L, CT>(CT(1), rho, ua, e);
        CT sn[NP + 1], dn[NP];
        sn[0] = f[0] - e[0];
        static_for<0, NP>([&](auto P) {
            constexpr int a = 2 * P + 1, b = a + 1;
            const CT na = f[a] - e[a], nb = f[b] - e[b];
            sn[P + 1] = na + nb;
            dn[P] = na - nb;
        });
        static_for<0, NP + 1>([&](auto R) {
            CT re = CT(0);
            static_for<0, NP + 1>([&](auto C_) { re += p.mrt_ce[k][R][C_] * sn[C_]; });
            if constexpr (R == 0) {
                f[0] -= re;
            } else {
                CT ro = CT(0);
                static_for<0, NP>([&](auto C_) { ro += p.mrt_co[k][R - 1][C_] * dn[C_]; });
                f[2 * R - 1] -= re + ro;
                f[2 * R] -= re - ro;
            }
        });
        if (!shift) {  // EDM source (Eq. 5)
            static_for<0, L::Q>([&](auto I) { f[I] -= e[I]; });
            add_feq<L, CT>(CT(1), rho, ub, f);
        }
    }
}

// which (dy,dz) rows of the 3x3 neighbourhood does the lattice touch, and with which dx
template <class L>
constexpr bool row_has(int dy, int dz, int dx) {
    for (int i = 1; i < L::Q; ++i)
        if (L::E[i][0] == dx && L::E[i][1] == dy && L::E[i][2] == dz) return true;
    return false;
}
template <class L>
constexpr int dir_of(int dx, int dy, int dz) {
    for (int i = 0; i < L::Q; ++i)
        if (L::E[i][0] == dx && L::E[i][1] == dy && L::E[i][2] == dz) return i;
    return -1;
}

// S4 sums for VEC cells: S[a][v] = sum_i (w_i/cs2) psi(x_v + e_i) e_ia  and psi at the cells themselves.
// rowfn(IC<dy>, IC<dz>, IC<need_x>, t, left, right) delivers psi of the row (y+dy, z+dz): t[v] at the thread's VEC
// cells and, when need_x, the values left of lane 0 / right of lane VEC-1 (global memory in K2, shared memory in K2F).
// S4 sums for VEC cells: S[a][v] = sum_i (w_i/cs2) psi(x_v + e_i) e_ia  and psi at the cells themselves.
// rowfn(IC<dy>, IC<dz>, IC<need_x>, t, left, right) delivers psi of the row (y+dy, z+dz): t[v] at the thread's VEC
// cells and, when need_x, the values left of lane 0 / right of lane VEC-1 (global memory in K2, shared memory in K2F).
template <class L, class CT, int VEC, class RowFn>
__device__ __forceinline__ void psi_sums_rows(RowFn&& rowfn, CT (&S)[3][VEC], CT (&pc)[VEC]) {
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int v = 0; v < VEC; ++v) S[a][v] = CT(0);
    static_for<0, 9>([&](auto RW) {
        constexpr int dy = RW % 3 - 1, dz = RW / 3 - 1;
        constexpr bool centre = dy == 0 && dz == 0;
        constexpr bool has0 = row_has<L>(dy, dz, 0), hasx = row_has<L>(dy, dz, 1);
        if constexpr ((has0 || hasx || centre) && (L::D == 3 || dz == 0)) {
            CT t[VEC], left = CT(0), right = CT(0);
            rowfn(IC<dy>{}, IC<dz>{}, IC<(hasx ? 1 : 0)>{}, t, left, right);
            if constexpr (centre) {
#pragma unroll
                for (int v = 0; v < VEC; ++v) pc[v] = t[v];
            }
            if constexpr (has0) {
                constexpr int i = dir_of<L>(0, dy, dz);
                constexpr CT gw = CT(3 * L::WN[i]) / CT(L::WD);
#pragma unroll
                for (int v = 0; v < VEC; ++v) {
                    if constexpr (dy != 0) S[1][v] += CT(gw * dy) * t[v];
                    if constexpr (dz != 0) S[2][v] += CT(gw * dz) * t[v];
                }
            }
            if constexpr (hasx) {
                constexpr int i = dir_of<L>(1, dy, dz);
                constexpr CT gw = CT(3 * L::WN[i]) / CT(L::WD);
#pragma unroll
                for (int v = 0; v < VEC; ++v) {
                    const CT m = v > 0 ? t[v - 1] : left;
                    const CT q = v < VEC - 1 ? t[v + 1] : right;
                    S[0][v] += gw * (q - m);
                    if constexpr (dy != 0) S[1][v] += CT(gw * dy) * (q + m);
                    if constexpr (dz != 0) S[2][v] += CT(gw * dz) * (q + m);
                }
            }
        }
    });
}

// ZC (Zhang-Chen weight, KParams::zc): the rows hold the signed root s; the sums use psi = max(s, 0) and
// Zs[a][v] = sum_i (w_i/cs2) U(x_v + e_i) e_ia with U = hg s |s| is accumulated as well.
template <class L, class CT, int VEC, bool ZC, class RowFn>
__device__ __forceinline__ void psi_sums_rows_zc(RowFn&& rowfn, CT (&S)[3][VEC], CT (&pc)[VEC], CT (*Zs)[VEC], CT hg) {
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int v = 0; v < VEC; ++v) {
            S[a][v] = CT(0);
            if constexpr (ZC) Zs[a][v] = CT(0);
        }
    auto accumulate = [&](auto DY, auto DZ, auto HAS0, auto HASX, const CT (&t)[VEC], CT left, CT right, CT (*acc)[VEC]) {
        constexpr int dy = DY, dz = DZ;
        if constexpr (HAS0 != 0) {
            constexpr int i = dir_of<L>(0, dy, dz);
            constexpr CT gw = CT(3 * L::WN[i]) / CT(L::WD);
#pragma unroll
            for (int v = 0; v < VEC; ++v) {
                if constexpr (dy != 0) acc[1][v] += CT(gw * dy) * t[v];
                if constexpr (dz != 0) acc[2][v] += CT(gw * dz) * t[v];
            }
        }
        if constexpr (HASX != 0) {
            constexpr int i = dir_of<L>(1, dy, dz);
            constexpr CT gw = CT(3 * L::WN[i]) / CT(L::WD);
#pragma unroll
            for (int v = 0; v < VEC; ++v) {
                const CT m = v > 0 ? t[v - 1] : left;
                const CT q = v < VEC - 1 ? t[v + 1] : right;
                acc[0][v] += gw * (q - m);
                if constexpr (dy != 0) acc[1][v] += CT(gw * dy) * (q + m);
                if constexpr (dz != 0) acc[2][v] += CT(gw * dz) * (q + m);
            }
        }
    };
    static_for<0, 9>([&](auto RW) {
        constexpr int dy = RW % 3 - 1, dz = RW / 3 - 1;
        constexpr bool centre = dy == 0 && dz == 0;
        constexpr bool has0 = row_has<L>(dy, dz, 0), hasx = row_has<L>(dy, dz, 1);
        if constexpr ((has0 || hasx || centre) && (L::D == 3 || dz == 0)) {
            CT t[VEC], left = CT(0), right = CT(0);
            rowfn(IC<dy>{}, IC<dz>{}, IC<(hasx ? 1 : 0)>{}, t, left, right);
            if constexpr (ZC) {
                CT u[VEC];
#pragma unroll
                for (int v = 0; v < VEC; ++v) { u[v] = hg * t[v] * fabs(t[v]); t[v] = t[v] > CT(0) ? t[v] : CT(0); }
                const CT ul = hg * left * fabs(left), ur = hg * right * fabs(right);
                left = left > CT(0) ? left : CT(0);
                right = right > CT(0) ? right : CT(0);
                accumulate(IC<dy>{}, IC<dz>{}, IC<(has0 ? 1 : 0)>{}, IC<(hasx ? 1 : 0)>{}, u, ul, ur, Zs);
            }
            if constexpr (centre) {
#pragma unroll
                for (int v = 0; v < VEC; ++v) pc[v] = t[v];
            }
            accumulate(IC<dy>{}, IC<dz>{}, IC<(has0 ? 1 : 0)>{}, IC<(hasx ? 1 : 0)>{}, t, left, right, S);
        }
    });
}

// psi rows from the global psi field (two-pass path)
template <class L, class CT, int VEC, bool ZC = false>
__device__ __forceinline__ void psi_sums_vec(const CT* __restrict__ ps, const VCell& c, CT (&S)[3][VEC], CT (&pc)[VEC],
                                             CT (*Zs)[VEC] = nullptr, CT hg = CT(0)) {
    auto rowfn = [&](auto DY, auto DZ, auto NX, CT (&t)[VEC], CT& left, CT& right) {
        const CT* row = ps + (c.zo[1 + DZ] + c.yo[1 + DY]);
        ld_vec<CT, CT, VEC>(row + c.x0, t);
        if constexpr (NX != 0) { left = __ldg(row + c.xm); right = __ldg(row + c.xp); }
    };
    if constexpr (ZC) psi_sums_rows_zc<L, CT, VEC, true>(rowfn, S, pc, Zs, hg);
    else psi_sums_rows<L, CT, VEC>(rowfn, S, pc);
}

// S4 + S5 for one cell: du^k = F^k / rho^k with F^k = -psi^k sum_k' g_kk' S^k' (Eq. 13, Eq. 5) and the common
// velocity u' (R6) from the moments.
// With a Zhang-Chen weight (Z != nullptr): F^k = (1 - A_kk) F_SC^k + A_kk F_ZC^k, F_ZC^k = -Z^k (Eq. 13).
template <int NC, class CT>
__device__ __forceinline__ void force_and_velocity(const KParams<CT>& p, const CT (&rho)[NC], const CT (&j)[NC][3],
                                                   const CT (&S)[NC][3], const CT (&pc)[NC], CT (&u)[3], CT (&du)[NC][3],
                                                   const CT (*Z)[3] = nullptr) {
    CT inv_r[NC];
#pragma unroll
    for (int k = 0; k < NC; ++k) {
        inv_r[k] = CT(1) / rho[k];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            CT acc = CT(0);
#pragma unroll
            for (int kp = 0; kp < NC; ++kp) acc += p.G[k][kp] * S[kp][a];
            CT F = -pc[k] * acc;
            if (Z != nullptr && p.zc[k]) F = (CT(1) - p.zcA[k]) * F - p.zcA[k] * Z[k][a];
            du[k][a] = F * inv_r[k] + p.body[a];   // body force rho^k a (R19)
        }
    }
    if constexpr (NC == 1) {
#pragma unroll
        for (int a = 0; a < 3; ++a) u[a] = j[0][a] * inv_r[0];
    } else {
        CT den = CT(0);
#pragma unroll
        for (int k = 0; k < NC; ++k) den += rho[k] * p.inv_tau[k];
        const CT inv_den = CT(1) / den;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            CT num = CT(0);
#pragma unroll
            for (int k = 0; k < NC; ++k) num += j[k][a] * p.inv_tau[k];
            u[a] = num * inv_den;
        }
    }
}

// Links of a fluid cell that cross a velocity / pressure face: the rule is applied at the writing cell (R10), on the
// post-collision populations fc of component k; uc = common velocity of the cell.  facefn(IC<o>) = the non-periodic face
// the link along +e_o crosses, or -1.
template <class L, class CT, class FaceFn>
__device__ __forceinline__ void apply_face_rules_fn(const KParams<CT>& p, FaceFn&& facefn, int k, const CT (&uc)[3], CT (&fc)[L::Q]) {
    const CT uu15 = CT(1.5) * (uc[0] * uc[0] + uc[1] * uc[1] + uc[2] * uc[2]);
    static_for<1, L::Q>([&](auto O) {
        constexpr int o = O;
        constexpr int eox = L::E[o][0], eoy = L::E[o][1], eoz = L::E[o][2];
        constexpr CT w = CT(L::WN[o]) / CT(L::WD);
        const int face = facefn(O);
        if (face >= 0) {
            const int kind = p.face_kind[face];
            if (kind == FACE_VELOCITY) {   // arriving direction i = opposite(o), e_i = -e_o
                CT eu = CT(0);
                if constexpr (eox != 0) eu -= CT(eox) * p.face_u[face][0];
                if constexpr (eoy != 0) eu -= CT(eoy) * p.face_u[face][1];
                if constexpr (eoz != 0) eu -= CT(eoz) * p.face_u[face][2];
                fc[o] = fc[o] + CT(2) * w * p.face_rho[face][k] * eu * CT(3);
            } else if (kind == FACE_PRESSURE) {
                CT eu = CT(0);
                if constexpr (eox != 0) eu += CT(eox) * uc[0];
                if constexpr (eoy != 0) eu += CT(eoy) * uc[1];
                if constexpr (eoz != 0) eu += CT(eoz) * uc[2];
                fc[o] = -fc[o] + CT(2) * w * p.face_rho[face][k] * (CT(1) + CT(4.5) * eu * eu - uu15);
            }
        }
    });
}
// ... with the face found from the cell's coordinates (dense layout)
template <class L, class CT>
__device__ __forceinline__ void apply_face_rules(const KParams<CT>& p, const Cell& cc, int k, const CT (&uc)[3], CT (&fc)[L::Q]) {
    apply_face_rules_fn<L, CT>(p, [&](auto O) { return crossed_face<L, decltype(O)::value>(p, cc); }, k, uc, fc);
}

// ------------------------------------------------------------------ K1: rho + psi
// LIST: thread t owns the fluid cell p.flist[t] (porous domains: the dense mapping leaves most lanes on solid cells)
// (one cell per thread -- list mode, ragged rows -- is latency-bound: cap the registers for four CTAs per SM)
template <class L, int NC, class CT, class ST, bool BND, int VEC, bool LIST = false>
__global__ void __launch_bounds__(256, (VEC == 1 ? 4 : 1)) k_moments_v(const __grid_constant__ KParams<CT> p) {
    static_assert(!LIST || (BND && VEC == 1), "list mode is one cell per thread on a masked domain");
    pdl_begin();
    unsigned vid = blockIdx.x * blockDim.x + threadIdx.x;
    if constexpr (LIST) {
        if (vid >= (unsigned)p.nfluid) return;
        vid = (unsigned)__ldg(p.flist + vid);
    } else {
        if (vid >= (unsigned)p.N / VEC) return;
    }
    const VCell c = make_vcell<L, VEC>(p, vid);
    uint32_t fl[VEC];
    if (!load_flags<BND, VEC>(p, c, fl)) return;
#pragma unroll
    for (int k = 0; k < NC; ++k) {
        CT f[L::Q][VEC];
        pull_vec<L, CT, ST, BND, VEC>(p, c, fl, k, f);
        CT r[VEC], ps[VEC];
#pragma unroll
        for (int v = 0; v < VEC; ++v) {
            CT fc[L::Q];
            static_for<0, L::Q>([&](auto I) { fc[I] = f[I][v]; });
            r[v] = density<L, CT>(fc);
            ps[v] = psi_of_rho(p, k, r[v]);
        }
        store_lanes<CT, CT, BND, VEC>(p.psi + (long long)k * p.N + c.id0, ps, fl);
        if (p.write_rho) store_lanes<CT, CT, BND, VEC>(p.rho + (long long)k * p.N + c.id0, r, fl);
    }
}

// ------------------------------------------------------------------ K2: fused stream + force + collide + boundary
// COLL: 0 BGK, 1 MRT, 2 none (LBM_FLAG_NO_COLLIDE: pure streaming)
// ZC: some component carries a Zhang-Chen weight A_kk != 0 (Eq. 11-13); built for VEC = 1 only
template <class L, int NC, class CT, class ST, int COLL, bool BND, int VEC, bool LIST = false, bool ZC = false>
__global__ void __launch_bounds__(128, ((LIST && sizeof(ST) == 2) ? 6 : 1)) k_step_v(const __grid_constant__ KParams<CT> p) {
    static_assert(!LIST || (BND && VEC == 1), "list mode is one cell per thread on a masked domain");
    static_assert(!ZC || (VEC == 1 && !LIST && COLL != 2), "the Zhang-Chen variant is one cell per thread");
    pdl_begin();
    unsigned vid = blockIdx.x * blockDim.x + threadIdx.x;
    if constexpr (LIST) {
        if (vid >= (unsigned)p.nfluid) return;
        vid = (unsigned)__ldg(p.flist + vid);
    } else {
        if (vid >= (unsigned)p.N / VEC) return;
    }
    const VCell c = make_vcell<L, VEC>(p, vid);
    uint32_t fl[VEC];
    if (!load_flags<BND, VEC>(p, c, fl)) return;

    // S7 (read side) + S1
    CT f[NC][L::Q][VEC], rho[NC][VEC], j[NC][3][VEC];
#pragma unroll
    for (int k = 0; k < NC; ++k) {
        pull_vec<L, CT, ST, BND, VEC>(p, c, fl, k, f[k]);
        if constexpr (COLL != 2) {
#pragma unroll
            for (int v = 0; v < VEC; ++v) {
                CT fc[L::Q], jj[3];
                static_for<0, L::Q>([&](auto I) { fc[I] = f[k][I][v]; });
                moments<L, CT>(fc, rho[k][v], jj);
                j[k][0][v] = jj[0]; j[k][1][v] = jj[1]; j[k][2][v] = jj[2];
            }
        }
    }

    CT u[3][VEC], du[NC][3][VEC];
    if constexpr (COLL != 2) {
        // S4: F^k = -psi^k(x) sum_k' g_kk' S^k'   (Eq. 13);  du = F / rho (Eq. 5)
        CT S[NC][3][VEC], pc[NC][VEC];
        CT Zs[ZC ? NC : 1][3][VEC];
#pragma unroll
        for (int kp = 0; kp < NC; ++kp) {
            if constexpr (ZC) psi_sums_vec<L, CT, VEC, true>(p.psi + (long long)kp * p.N, c, S[kp], pc[kp], Zs[kp], p.zc_hg[kp]);
            else psi_sums_vec<L, CT, VEC>(p.psi + (long long)kp * p.N, c, S[kp], pc[kp]);
        }
#pragma unroll
        for (int v = 0; v < VEC; ++v) {
            CT rc[NC], jc[NC][3], Sc[NC][3], pcc[NC], uc[3], duc[NC][3];
            CT Zc[NC][3];
#pragma unroll
            for (int k = 0; k < NC; ++k) {
                rc[k] = rho[k][v];
                pcc[k] = pc[k][v];
#pragma unroll
                for (int a = 0; a < 3; ++a) {
                    jc[k][a] = j[k][a][v]; Sc[k][a] = S[k][a][v];
                    if constexpr (ZC) Zc[k][a] = Zs[k][a][v];
                }
            }
            if constexpr (ZC) force_and_velocity<NC, CT>(p, rc, jc, Sc, pcc, uc, duc, Zc);
            else force_and_velocity<NC, CT>(p, rc, jc, Sc, pcc, uc, duc);
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                u[a][v] = uc[a];
#pragma unroll
                for (int k = 0; k < NC; ++k) du[k][a][v] = duc[k][a];
            }
        }
    } else {
#pragma unroll
        for (int a = 0; a < 3; ++a)
#pragma unroll
            for (int v = 0; v < VEC; ++v) u[a][v] = CT(0);
    }

    // S6 + S7 (write side)
#pragma unroll
    for (int k = 0; k < NC; ++k) {
#pragma unroll
        for (int v = 0; v < VEC; ++v) {
            if (BND && (fl[v] & SOLID_BIT)) continue;
            CT fc[L::Q];
            static_for<0, L::Q>([&](auto I) { fc[I] = f[k][I][v]; });
            const CT uc[3] = {u[0][v], u[1][v], u[2][v]};
            if constexpr (COLL != 2) {
                const CT dc[3] = {du[k][0][v], du[k][1][v], du[k][2][v]};
                collide<L, COLL, CT>(p, k, rho[k][v], uc, dc, fc);
                // Surface-tension control (Eq. 14-16; D2Q9 MRT, reading R20): source C in moment space from
                // Q = kappa g_kk [(1-A) psi sum_i G_i (psi(x+e_i) - psi) e_i e_i + (A/2) sum_i G_i (psi(x+e_i)^2 - psi^2) e_i e_i]
                if constexpr (ZC && L::D == 2 && COLL == 1) {
                    if (p.st_on[k]) {
                        const CT* ps = p.psi + (long long)k * p.N;
                        auto pos = [&](CT s_) { return (p.zc[k] && s_ < CT(0)) ? CT(0) : s_; };
                        const CT ps0 = pos(__ldg(ps + c.yo[1] + c.x0));
                        const CT A = p.zcA[k];
                        CT Qxx = CT(0), Qyy = CT(0), Qxy = CT(0);
                        static_for<1, L::Q>([&](auto I) {
                            constexpr int i = I;
                            constexpr int ex = L::E[i][0], ey = L::E[i][1];
                            constexpr CT gw = CT(3 * L::WN[i]) / CT(L::WD);
                            const CT ps1 = pos(__ldg(ps + c.yo[1 + ey] + (ex == 0 ? c.x0 : (ex > 0 ? c.xp : c.xm))));
                            const CT t = gw * ((CT(1) - A) * ps0 * (ps1 - ps0) + CT(0.5) * A * (ps1 * ps1 - ps0 * ps0));
                            if constexpr (ex != 0) Qxx += t;
                            if constexpr (ey != 0) Qyy += t;
                            if constexpr (ex * ey != 0) Qxy += CT(ex * ey) * t;
                        });
                        // C_r (Eq. 15) for the moments e, eps, pxx, pxy; st_coef = kappa g_kk {1.5 s_e, -1.5 s_eps, -s_nu, -s_nu}
                        const CT C1 = p.st_coef[k][0] * (Qxx + Qyy), C2 = p.st_coef[k][1] * (Qxx + Qyy);
                        const CT C7 = p.st_coef[k][2] * (Qxx - Qyy), C8 = p.st_coef[k][3] * Qxy;
                        static_for<0, L::Q>([&](auto I) {   // f* += M^-1 C,  M^-1 = M^T diag(1 / |row|^2) (R9)
                            constexpr int i = I;
                            fc[i] += C1 * (CT(mrt_entry<L>(1, i)) / CT(mrt_norm2<L>(1))) + C2 * (CT(mrt_entry<L>(2, i)) / CT(mrt_norm2<L>(2))) +
                                     C7 * (CT(mrt_entry<L>(7, i)) / CT(mrt_norm2<L>(7))) + C8 * (CT(mrt_entry<L>(8, i)) / CT(mrt_norm2<L>(8)));
                        });
                    }
                }
            }
            // links across velocity / pressure faces: the rule is applied at the writing cell (R10)
            if constexpr (BND) {
                if (fl[v] & FACEBC_BIT) {
                    Cell cc;
                    cc.x = c.x0 + v; cc.y = c.y; cc.z = c.z;
                    apply_face_rules<L, CT>(p, cc, k, uc, fc);
                }
            }
            static_for<0, L::Q>([&](auto I) { f[k][I][v] = fc[I] - p.wref[I]; });
        }
        ST* out = static_cast<ST*>(p.f_out) + (long long)k * L::Q * p.plane + c.id0;
        static_for<0, L::Q>([&](auto I) { store_lanes<CT, ST, BND, VEC>(out + (long long)I * p.plane, f[k][I], fl); });
    }
}

}  // namespace lbmk
