// lbm_fused.cuh -- K2F, the one-pass hot kernel of the Shan-Chen LBM step for sm_100a (fully periodic domains
// without solid cells).
//
//   k_fused_v   S1 (rho, j) + S3 (psi) + S4..S7 in ONE pass over the populations
//               Eq. 4/10, Eq. 12, Eq. 13, Eq. 3, Eq. 5, Eq. 2
//
// Why: the two-pass path (K1 then K2, lbm_hot.cuh) runs at the speed of a copy, so the only way up is to move
// fewer bytes: B2 = 3 q s + 2 c per cell against B1 = 2 q s for one pass.  The force needs psi(rho)
// of the NEW time level at the 18 (8) neighbours, which is what forced the separate K1 pass.  K2F instead
// recomputes rho -> psi of a one-cell ring around its tile from the populations themselves:
//
//   * a CTA owns an x-y tile of TX x TY cells and marches along z over `mchunk` planes (D2Q9: a strip of TX cells
//     marching along y).  One warp per tile row; every lane owns VEC consecutive cells (128/64-bit accesses).
//   * marching step m: the warp pulls the populations of plane m+1 of its row (S7 read side), sums rho, evaluates
//     psi and writes it to a 4-slot ring of psi planes in shared memory; two extra "halo" warps do the same for the
//     rows just outside the tile and the edge lanes for the two columns left / right of it (scalar loads).  After
//     one __syncthreads the interior warps collide plane m (its populations were pulled one step earlier and
//     carried in registers) with the force taken from the psi planes m-1, m, m+1 in shared memory, and store.
//   * the ring re-reads (TY+2)/TY of the populations, but those re-reads are L2 hits (the neighbouring CTA reads
//     the same lines at about the same time): DRAM traffic stays ~ 2 q s per cell.
//   * the next plane is prefetched into L2 while the current one is collided, so one CTA per SM is enough to keep
//     HBM busy although the CTA works in phases.
// The psi tiles never exist in global memory, so there is nothing for TMA to stage (north_star's "TMA where the
// tile shape allows" applied to the two-pass psi field).  Arithmetic is shared with K2 (lbm_hot.cuh), in the
// same order.
#pragma once
#include "lbm_hot.cuh"

namespace lbmk {

template <class L, int NC, class CT, int VEC, int WX, int TY>
struct FusedTile {
    static constexpr int HR = L::D == 3 ? 1 : 0;      // halo rows on each side of the tile (none in 2-D)
    static constexpr int ROWS = TY + 2 * HR;
    static constexpr int TX = WX * 32 * VEC;
    static constexpr int PAD = 16 / (int)sizeof(CT);  // cells left of the tile in a shared row (keeps vectors aligned)
    static constexpr int PITCH = TX + 2 * PAD;
    static constexpr int SLOTS = 4;
    static constexpr int THREADS = WX * ROWS * 32;
    static constexpr size_t SMEM = sizeof(CT) * NC * SLOTS * ROWS * PITCH;
    static_assert(L::D == 3 || TY == 1, "2-D tiles are one row (the march runs along y)");
    static_assert(SMEM <= 48 * 1024, "psi ring must fit static shared memory");
    static_assert(THREADS <= 1024, "CTA too large");
};

__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

// mchunk: planes (3-D: z, 2-D: y rows) marched by one CTA.  PF: prefetch plane m+2 into L2 while plane m collides.
template <class L, int NC, class CT, class ST, int COLL, int VEC, int WX, int TY, bool PF>
__global__ void __launch_bounds__(FusedTile<L, NC, CT, VEC, WX, TY>::THREADS, 1)
k_fused_v(const __grid_constant__ KParams<CT> p, int mchunk) {
    using T = FusedTile<L, NC, CT, VEC, WX, TY>;
    constexpr bool D3 = L::D == 3;
    constexpr int Q = L::Q;
    __shared__ __align__(16) CT psi_s[NC][T::SLOTS][T::ROWS][T::PITCH];

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int r = warp / WX;                                   // tile row of this warp
    const int xl = ((warp % WX) * 32 + lane) * VEC;            // first cell of this lane inside the tile
    const int tx0 = blockIdx.x * T::TX;
    const int txw = min(T::TX, p.nx - tx0);                    // tile width (nx % VEC == 0)
    const int nm = D3 ? p.nz : p.ny;                           // extent of the marching axis
    const int mstride = D3 ? p.nx * p.ny : p.nx;
    const int m0 = (D3 ? blockIdx.z : blockIdx.y) * mchunk;
    const int m1 = min(nm, m0 + mchunk);

    // rows of the tile: r = 0 and r = nint+1 are the halo rows (3-D only)
    bool used = true, interior = true;
    int yw = 0;
    if constexpr (D3) {
        const int yb = blockIdx.y * TY;
        const int nint = min(TY, p.ny - yb);
        used = r <= nint + 1;
        interior = r >= 1 && r <= nint;
        const int yy = yb - 1 + r;
        yw = yy < 0 ? yy + p.ny : (yy >= p.ny ? yy - p.ny : yy);
    }
    const bool act = used && xl < txw;
    const bool ring_l = act && xl == 0, ring_r = act && xl + VEC == txw;

    // geometry of the thread's cells and of the two ring cells of its row; the marching offsets are filled per plane
    VCell c, cl, cr;
    c.x0 = tx0 + xl;
    c.xm = c.x0 > 0 ? c.x0 - 1 : p.nx - 1;
    c.xp = c.x0 + VEC < p.nx ? c.x0 + VEC : 0;
    cl.x0 = tx0 > 0 ? tx0 - 1 : p.nx - 1;
    cr.x0 = tx0 + txw < p.nx ? tx0 + txw : 0;
    cl.xm = cl.x0 > 0 ? cl.x0 - 1 : p.nx - 1;
    cl.xp = cl.x0 + 1 < p.nx ? cl.x0 + 1 : 0;
    cr.xm = cr.x0 > 0 ? cr.x0 - 1 : p.nx - 1;
    cr.xp = cr.x0 + 1 < p.nx ? cr.x0 + 1 : 0;
    c.y = yw; c.z = 0; c.id0 = 0;
    if constexpr (D3) {
        c.yo[1] = yw * p.nx;
        c.yo[0] = (yw > 0 ? yw - 1 : p.ny - 1) * p.nx;
        c.yo[2] = (yw < p.ny - 1 ? yw + 1 : 0) * p.nx;
    } else {
        c.zo[0] = c.zo[1] = c.zo[2] = 0;
    }
    auto wrap_m = [&](int m) { return m < 0 ? m + nm : (m >= nm ? m - nm : m); };
    // offsets of planes ml-1, ml, ml+1 along the marching axis
    auto set_plane = [&](int ml) {
        const int a = wrap_m(ml - 1) * mstride, b = wrap_m(ml) * mstride, d = wrap_m(ml + 1) * mstride;
        if constexpr (D3) { c.zo[0] = a; c.zo[1] = b; c.zo[2] = d; }
        else { c.yo[0] = a; c.yo[1] = b; c.yo[2] = d; }
    };
    const uint32_t nofl[VEC] = {};
    const uint32_t nofl1[1] = {0};

    // S7 read side + S1 (rho) + S3 for plane ml: populations into f (kept by the interior warps), psi into slot
    auto load_plane = [&](int ml, CT (&f)[NC][Q][VEC]) {
        set_plane(ml);
        const int slot = (ml + 4) & 3;
        if (act) {
#pragma unroll
            for (int k = 0; k < NC; ++k) {
                pull_vec<L, CT, ST, false, VEC>(p, c, nofl, k, f[k]);
                CT ps[VEC];
#pragma unroll
                for (int v = 0; v < VEC; ++v) {
                    CT fc[Q];
                    static_for<0, Q>([&](auto I) { fc[I] = f[k][I][v]; });
                    ps[v] = psi_of_rho(p, k, density<L, CT>(fc));
                }
                st_vec<CT, CT, VEC>(&psi_s[k][slot][r][T::PAD + xl], ps);
            }
            if (ring_l | ring_r) {
#pragma unroll
                for (int side = 0; side < 2; ++side) {
                    if (side == 0 ? ring_l : ring_r) {
                        VCell e = c;
                        e.x0 = side == 0 ? cl.x0 : cr.x0;
                        e.xm = side == 0 ? cl.xm : cr.xm;
                        e.xp = side == 0 ? cl.xp : cr.xp;
#pragma unroll
                        for (int k = 0; k < NC; ++k) {
                            CT g[Q][1], fc[Q];
                            pull_vec<L, CT, ST, false, 1>(p, e, nofl1, k, g);
                            static_for<0, Q>([&](auto I) { fc[I] = g[I][0]; });
                            psi_s[k][slot][r][side == 0 ? T::PAD - 1 : T::PAD + txw] = psi_of_rho(p, k, density<L, CT>(fc));
                        }
                    }
                }
            }
        }
    };

    // L2 prefetch of the lines the thread will pull for plane ml
    auto prefetch_plane = [&](int ml) {
        if (!act) return;
        const int a = wrap_m(ml - 1) * mstride, b = wrap_m(ml) * mstride, d = wrap_m(ml + 1) * mstride;
#pragma unroll
        for (int k = 0; k < NC; ++k) {
            const ST* base = static_cast<const ST*>(p.f_in) + (long long)k * Q * p.plane;
            static_for<0, Q>([&](auto I) {
                constexpr int i = I;
                constexpr int ey = L::E[i][1], ez = L::E[i][2];
                int off;
                if constexpr (D3) off = (ez > 0 ? a : (ez < 0 ? d : b)) + c.yo[1 - ey];
                else off = (ey > 0 ? a : (ey < 0 ? d : b));
                prefetch_l2(base + (long long)i * p.plane + off + c.x0);
            });
        }
    };

    // S1 (j) + S4..S6 + S7 write side for plane m of the thread's cells
    auto collide_plane = [&](int m, CT (&f)[NC][Q][VEC]) {
        const int sc = (m + 4) & 3;
        CT S[NC][3][VEC], pc[NC][VEC];
        if constexpr (COLL != 2) {
#pragma unroll
            for (int kp = 0; kp < NC; ++kp) {
                psi_sums_rows<L, CT, VEC>(
                    [&](auto DY, auto DZ, auto NX, CT (&t)[VEC], CT& left, CT& right) {
                        const CT* row;
                        if constexpr (D3) row = &psi_s[kp][(sc + DZ + 4) & 3][r + DY][T::PAD + xl];
                        else row = &psi_s[kp][(sc + DY + 4) & 3][0][T::PAD + xl];
                        using R = typename RawVec<sizeof(CT) * VEC>::type;
                        const R raw = *reinterpret_cast<const R*>(row);
                        const CT* tv = reinterpret_cast<const CT*>(&raw);
#pragma unroll
                        for (int v = 0; v < VEC; ++v) t[v] = tv[v];
                        if constexpr (NX != 0) { left = row[-1]; right = row[VEC]; }
                    },
                    S[kp], pc[kp]);
            }
        }
        const int id0 = wrap_m(m) * mstride + (D3 ? yw * p.nx : 0) + c.x0;
#pragma unroll
        for (int v = 0; v < VEC; ++v) {
            CT fc[NC][Q];
#pragma unroll
            for (int k = 0; k < NC; ++k) static_for<0, Q>([&](auto I) { fc[k][I] = f[k][I][v]; });
            if constexpr (COLL != 2) {
                CT rc[NC], jc[NC][3], Sc[NC][3], pcc[NC], uc[3], duc[NC][3];
#pragma unroll
                for (int k = 0; k < NC; ++k) {
                    moments<L, CT>(fc[k], rc[k], jc[k]);
                    pcc[k] = pc[k][v];
#pragma unroll
                    for (int a = 0; a < 3; ++a) Sc[k][a] = S[k][a][v];
                }
                force_and_velocity<NC, CT>(p, rc, jc, Sc, pcc, uc, duc);
#pragma unroll
                for (int k = 0; k < NC; ++k) collide<L, COLL, CT>(p, k, rc[k], uc, duc[k], fc[k]);
            }
#pragma unroll
            for (int k = 0; k < NC; ++k) static_for<0, Q>([&](auto I) { f[k][I][v] = fc[k][I] - p.wref[I]; });
        }
#pragma unroll
        for (int k = 0; k < NC; ++k) {
            ST* out = static_cast<ST*>(p.f_out) + (long long)k * Q * p.plane + id0;
            static_for<0, Q>([&](auto I) { st_vec<CT, ST, VEC>(out + (long long)I * p.plane, f[k][I]); });
        }
    };

    CT A[NC][Q][VEC], B[NC][Q][VEC];
    load_plane(m0 - 1, B);   // psi only
    load_plane(m0, A);
    if constexpr (PF) prefetch_plane(m0 + 1);
    for (int m = m0; m < m1; ++m) {
        load_plane(m + 1, B);
        if constexpr (PF) {
            if (m + 2 <= m1) prefetch_plane(m + 2);
        }
        __syncthreads();
        if (interior && act) collide_plane(m, A);
#pragma unroll
        for (int k = 0; k < NC; ++k)
            static_for<0, Q>([&](auto I) {
#pragma unroll
                for (int v = 0; v < VEC; ++v) A[k][I][v] = B[k][I][v];
            });
    }
}

}  // namespace lbmk
