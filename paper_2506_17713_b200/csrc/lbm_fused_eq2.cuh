// lbm_fused_eq2.cuh -- k_fused_eq with the row pipeline cut in two: a FRONT warp and a BACK warp per tile row.
//
//   k_fused_eq_split   same step, same tiles and same arithmetic as k_fused_eq (lbm_fused_eq.cuh; S1 + S3 + S4..S7 for one
//                      component, BGK with tau = 1), other schedule.
//
// In k_fused_eq one warp per row does everything for a plane in turn -- shared-memory loads and moments of plane pl,
// then force, equilibrium and the 19 stores of the pending plane pl-1 -- and all rows meet at the psi ring once per
// plane, so the eight warps of the SM are in the same phase at any time: while they store, no arithmetic is issued, and
// while they sum, the store path idles (copies alone 1.9 ms, + arithmetic 2.9 ms, + stores 3.9 ms on C5-512).  Here
//
//   front warp of row r, plane pl:  wait for the row's copies -> registers -> rho, j (S1) -> issue the copies of plane
//                                   pl+2 into the freed slot -> psi(rho) to the psi ring -> rho, j to the row's hand-over
//                                   slot (one slot of 16 bytes per cell; the values wait in registers until the back warp
//                                   has taken those of plane pl-1)
//   back warp of row r, plane pl-1: wait until the ring holds psi of plane pl -> take rho, j -> force (S4, S5),
//                                   f_eq(rho, u' + du) (S6) and store (S7 write side), in two halves of the row so that
//                                   38 instead of 76 output values are live
//
// The front warps run one to two planes ahead of the back warps; loads and sums of plane pl+1 overlap with the stores of
// plane pl-1.  The halo rows keep a single landing slot (they only sum rho; the hand-over slots take their second one)
// and hold the next plane's rho in registers instead.
// EARLY (template): the back warp takes rho, j BEFORE it waits for psi, which frees the hand-over slot a plane earlier and
// lets the front warps run further ahead.  Faster where the copies are not the bound (256^3: 0.51 -> 0.46 ms); on 384^3
// and 512^3 the rows of neighbouring tiles then drift apart, the halo rows they share leave L2 between the two reads
// (DRAM reads 11.5 -> 12.7 GB per step on 512^3; k_fused_eq: 10.6) and the step gets slower (4.0 -> 4.14 ms; k_fused_eq:
// 3.90): plan_fused (lbm_api.cu) picks the kernel per domain.  Stores carry an evict-first L2 policy: written lines are
// never read again within the step and would otherwise push the shared halo rows out (512^3: 4.1 -> 4.0 ms).  The same
// hint on the loads of the rows no other tile reads made it slower (4.3 ms) and is not used.
#pragma once
#include "lbm_fused_eq.cuh"

namespace lbmk {

// N values of a shared-memory row as one vector load
template <class CT, int N>
__device__ __forceinline__ void lds_vec(const CT* row, CT (&out)[N]) {
    using R = typename RawVec<sizeof(CT) * N>::type;
    const R raw = *reinterpret_cast<const R*>(row);
    const CT* tv = reinterpret_cast<const CT*>(&raw);
#pragma unroll
    for (int v = 0; v < N; ++v) out[v] = tv[v];
}

// L2 eviction policy (createpolicy) and the hinted form of the vector store
__device__ __forceinline__ uint64_t l2_evict_first() {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
template <class CT, class ST, int VEC>
__device__ __forceinline__ void st_vec_global_hint(ST* p, const CT (&in)[VEC], uint64_t pol) {
    using R = typename RawVec<sizeof(ST) * VEC>::type;
    R r;
    ST* t = reinterpret_cast<ST*>(&r);
#pragma unroll
    for (int v = 0; v < VEC; ++v) t[v] = Cvt<CT, ST>::down(in[v]);
    if constexpr (sizeof(R) == 16) {
        const uint4 u = *reinterpret_cast<const uint4*>(&r);
        asm volatile("st.global.L2::cache_hint.v4.b32 [%0], {%1, %2, %3, %4}, %5;" ::"l"(p), "r"(u.x), "r"(u.y), "r"(u.z), "r"(u.w), "l"(pol)
                     : "memory");
    } else if constexpr (sizeof(R) == 8) {
        const uint2 u = *reinterpret_cast<const uint2*>(&r);
        asm volatile("st.global.L2::cache_hint.v2.b32 [%0], {%1, %2}, %3;" ::"l"(p), "r"(u.x), "r"(u.y), "l"(pol) : "memory");
    } else if constexpr (sizeof(R) == 4) {
        const uint32_t u = *reinterpret_cast<const uint32_t*>(&r);
        asm volatile("st.global.L2::cache_hint.b32 [%0], %1, %2;" ::"l"(p), "r"(u), "l"(pol) : "memory");
    } else {
        const unsigned short u = *reinterpret_cast<const unsigned short*>(&r);
        asm volatile("st.global.L2::cache_hint.b16 [%0], %1, %2;" ::"l"(p), "h"(u), "l"(pol) : "memory");
    }
}

template <class L, class CT, class ST, int VEC, int TY>
struct EqSplitTile {
    static_assert(L::D == 3, "the kernel marches along z");
    static_assert(VEC % 2 == 0, "the back warps take a row in two halves");
    static constexpr int Q = L::Q;
    static constexpr int NSTG = 2;                                  // landing slots per interior row
    static constexpr int NS = 4;                                    // psi ring slots
    static constexpr int ROWS = TY + 2;
    static constexpr int TX = 32 * VEC;
    static constexpr int PAD = 16 / (int)sizeof(CT);
    static constexpr int PITCH = TX + 2 * PAD;
    static constexpr int PADS = 16 / (int)sizeof(ST);
    static constexpr int dir_pitch(int i) { return TX + (L::E[i][0] != 0 ? PADS : 0); }
    static constexpr int dir_lead(int i) { return L::E[i][0] > 0 ? PADS : 0; }
    static constexpr int dir_off(int i) { int o = 0; for (int j = 0; j < i; ++j) o += dir_pitch(j); return o; }
    static constexpr int RB = dir_off(Q);
    static constexpr int NCW = (TY + 3) / 4 * 4;                    // warps of the front group, and of the back group
    static constexpr int NPW = 4;                                   // two halo rows, two ring columns
    static constexpr int NPSI = TY + 4;                             // arrivals per psi plane
    static constexpr int THREADS = (2 * NCW + NPW) * 32;
    static constexpr size_t STAGE_ELEMS = (size_t)RB * TY;
    static constexpr size_t PSI_ELEMS = (size_t)NS * ROWS * PITCH;
    static constexpr size_t MOM_ELEMS = (size_t)TY * 4 * TX;        // rho, jx, jy, jz of one plane
    static constexpr int NBAR = NSTG * ROWS + 2 * NS + 2 * TY;
    static constexpr size_t SMEM = sizeof(ST) * (NSTG * STAGE_ELEMS + 2 * (size_t)RB) + sizeof(CT) * (PSI_ELEMS + MOM_ELEMS) + 8 * NBAR;
    static constexpr int REG_LAUNCH = (65536 / THREADS) / 8 * 8;
    static constexpr int REG_PROD = 40;
    static constexpr int REG_FRONT = 104;
    static constexpr int REG_BACK = ((REG_LAUNCH * THREADS - REG_PROD * NPW * 32 - REG_FRONT * NCW * 32) / (NCW * 32)) / 8 * 8;
    static constexpr long long REGS_NEEDED = (long long)REG_PROD * NPW * 32 + (long long)(REG_FRONT + REG_BACK) * NCW * 32;
    static_assert(SMEM <= 227 * 1024, "tile does not fit shared memory");
    static_assert(ROWS <= 32, "ring warps map one lane to one row");
};

template <class L, class CT, class ST, int VEC, int TY, bool EARLY, bool WREF>
__global__ void __launch_bounds__((EqSplitTile<L, CT, ST, VEC, TY>::THREADS), 1)
k_fused_eq_split(const __grid_constant__ KParams<CT> p, int mchunk, int yoff, int zoff) {
    using T = EqSplitTile<L, CT, ST, VEC, TY>;
    constexpr int Q = L::Q, NSTG = T::NSTG, NS = T::NS;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    ST* stage = reinterpret_cast<ST*>(smem_raw);                          // [NSTG][TY][RB]
    ST* halo = stage + NSTG * T::STAGE_ELEMS;                              // [2][RB]
    CT* psi_s = reinterpret_cast<CT*>(halo + 2 * T::RB);                   // [NS][ROWS][PITCH]
    CT* mom_s = psi_s + T::PSI_ELEMS;                                      // [TY][4][TX]
    uint64_t* bar_land = reinterpret_cast<uint64_t*>(mom_s + T::MOM_ELEMS);   // [NSTG][ROWS] copies of a row landed
    uint64_t* bar_psi = bar_land + NSTG * T::ROWS;                         // [NS] psi of a plane complete
    uint64_t* bar_free = bar_psi + NS;                                     // [NS] ring slot read for the last time
    uint64_t* bar_mf = bar_free + NS;                                      // [TY] hand-over slot of a row filled
    uint64_t* bar_me = bar_mf + TY;                                        // [TY] ... and taken

    const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
    const int lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int s = 0; s < NSTG * T::ROWS; ++s) mbar_init(bar_land + s, 1);
        for (int s = 0; s < NS; ++s) { mbar_init(bar_psi + s, T::NPSI); mbar_init(bar_free + s, TY); }
        for (int s = 0; s < 2 * TY; ++s) mbar_init(bar_mf + s, 1);
    }
    __syncthreads();

    const int tx0 = blockIdx.x * T::TX;
    const int txw = min(T::TX, p.nx - tx0);
    const int yb = ((int)blockIdx.y + yoff) * TY;      // (yoff, zoff: the launch covers a group of tile rows / one chunk of planes)
    const int nint = min(TY, p.ny - yb);
    const int nm = p.nz;
    const unsigned sy = (unsigned)p.nx, sz = (unsigned)p.nx * (unsigned)p.ny;
    const int m0 = ((int)blockIdx.z + zoff) * mchunk, m1 = min(nm, m0 + mchunk);
    const int nit = m1 - m0 + 2;                          // planes m0-1 .. m1 pass through the pipeline (it = 0 .. nit-1)
    const unsigned plane = (unsigned)p.plane;
    auto wrap_y = [&](int y) { return y < 0 ? y + p.ny : (y >= p.ny ? y - p.ny : y); };
    auto wrap_m = [&](int m) { return m < 0 ? m + nm : (m >= nm ? m - nm : m); };
    auto psi_row = [&](int slot, int r) { return psi_s + ((size_t)slot * T::ROWS + r) * T::PITCH; };
    const ST* fin = static_cast<const ST*>(p.f_in);

    // ---- bulk copies of tile row r, plane it (as in k_fused_eq: lane i < Q issues direction i)
    struct RowPipe {
        unsigned base_l;
        int ex_l, ez_l, off_l;
    };
    constexpr int NXD = []() { int n = 0; for (int i = 0; i < Q; ++i) n += L::E[i][0] != 0; return n; }();
    const uint32_t main_bytes = (uint32_t)txw * (uint32_t)sizeof(ST);
    const uint32_t land_bytes = (uint32_t)Q * main_bytes + (uint32_t)NXD * 16u;
    auto make_pipe = [&](int r) {
        RowPipe rp;
        int ex_l = 0, ey_l = 0, ez_l = 0, off_l = 0;
        static_for<0, Q>([&](auto I) {
            constexpr int ex = L::E[I][0], ey = L::E[I][1], ez = L::E[I][2], so = T::dir_off(I);
            if (lane == I) { ex_l = ex; ey_l = ey; ez_l = ez; off_l = so; }
        });
        const int yw = wrap_y(yb - 1 + r);
        rp.base_l = (unsigned)lane * plane + (unsigned)wrap_y(yw - ey_l) * sy;
        rp.ex_l = ex_l; rp.ez_l = ez_l; rp.off_l = off_l;
        return rp;
    };
    const int xlp = (tx0 > 0 ? tx0 : p.nx) - T::PADS;
    const int xrp = tx0 + txw < p.nx ? tx0 + txw : 0;
    auto issue = [&](const RowPipe& rp, int r, int it, ST* land) {
        uint64_t* lb = bar_land + (it & 1) * T::ROWS + r;
        if (lane == 0) mbar_expect_tx(lb, land_bytes);
        __syncwarp();
        if (lane < Q) {
            const int pl = m0 - 1 + it;
            const ST* src = fin + (rp.base_l + (unsigned)wrap_m(pl - rp.ez_l) * sz);
            ST* dst = land + rp.off_l;
            if (rp.ex_l > 0) {
                if (tx0 > 0) bulk_g2s(dst, src + (tx0 - T::PADS), main_bytes + 16u, lb);
                else { bulk_g2s(dst + T::PADS, src + tx0, main_bytes, lb); bulk_g2s(dst, src + xlp, 16u, lb); }
            } else if (rp.ex_l < 0) {
                if (tx0 + txw < p.nx) bulk_g2s(dst, src + tx0, main_bytes + 16u, lb);
                else { bulk_g2s(dst, src + tx0, main_bytes, lb); bulk_g2s(dst + txw, src + xrp, 16u, lb); }
            } else {
                bulk_g2s(dst, src + tx0, main_bytes, lb);
            }
        }
    };
    // a ring slot is rewritten with plane `it` once the back warps have read plane it-NS for the last time
    auto wait_free = [&](int it) {
        if (it >= NS) mbar_wait(bar_free + it % NS, (it / NS - 1) & 1);
    };

    // =============================================================== front: copies -> rho, j -> psi, hand-over
    auto front_role = [&]() {
        const int cw = warp, r = cw + 1;
        const int xl = lane * VEC;
        const bool used = cw < nint;
        const bool act = used && xl < txw;
        auto slot_of = [&](int it) { return stage + (size_t)(it & 1) * T::STAGE_ELEMS + (size_t)cw * T::RB; };
        const RowPipe rp = make_pipe(r);
        CT* mrow = mom_s + (size_t)cw * 4 * T::TX + xl;
        if (used) {
            issue(rp, r, 0, slot_of(0));
            issue(rp, r, 1, slot_of(1));
        }
        for (int it = 0; it < nit; ++it) {
            CT rho[VEC], j[3][VEC];
            if (used) mbar_wait(bar_land + (it & 1) * T::ROWS + r, (it >> 1) & 1);
            if (act) {
                CT A[Q][VEC];
                const ST* rows = slot_of(it) + xl;
                static_for<0, Q>([&](auto I) {
                    constexpr int i = I;
                    constexpr int so = T::dir_off(i) + T::dir_lead(i);
                    pulled_from_row<CT, ST, VEC, L::E[i][0]>(rows + so, A[i]);
                });
#pragma unroll
                for (int v = 0; v < VEC; ++v) {
                    CT fc[Q], jj[3];
                    static_for<0, Q>([&](auto I) {
                        if constexpr (WREF) fc[I] = A[I][v] + p.wref[I];
                        else fc[I] = A[I][v];
                    });
                    moments<L, CT>(fc, rho[v], jj);
                    j[0][v] = jj[0]; j[1][v] = jj[1]; j[2][v] = jj[2];
                }
            }
            __syncwarp();                                   // every lane has its values: the slot can be overwritten
            if (used && it + 2 < nit) issue(rp, r, it + 2, slot_of(it));
            wait_free(it);
            if (act) {
                CT ps[VEC];
#pragma unroll
                for (int v = 0; v < VEC; ++v) ps[v] = psi_of_rho(p, 0, rho[v]);
                st_vec<CT, CT, VEC>(psi_row(it % NS, r) + T::PAD + xl, ps);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_psi + it % NS);
            // hand-over h = it-1 of rho, j (planes 1 .. nit-2 are collided)
            if (used && it >= 1 && it + 1 < nit) {
                const int h = it - 1;
                if (h >= 1) mbar_wait(bar_me + cw, (h - 1) & 1);
                if (act) {
                    st_vec<CT, CT, VEC>(mrow, rho);
                    st_vec<CT, CT, VEC>(mrow + T::TX, j[0]);
                    st_vec<CT, CT, VEC>(mrow + 2 * T::TX, j[1]);
                    st_vec<CT, CT, VEC>(mrow + 3 * T::TX, j[2]);
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(bar_mf + cw);
            }
        }
    };

    // =============================================================== back: force, equilibrium, store of the pending plane
    auto back_role = [&]() {
        const int cw = warp - T::NCW;
        const bool used = cw < nint;
        const unsigned row0 = (unsigned)wrap_y(yb + cw) * sy + (unsigned)tx0;
        const CT* mrow = mom_s + (size_t)cw * 4 * T::TX;
        const uint64_t spol = l2_evict_first();
        for (int it = 2; it < nit; ++it) {
            CT prho[2][VEC / 2], pj[2][3][VEC / 2];
            auto take = [&]() {                            // rho, j of the pending plane it-1 out of the hand-over slot
                mbar_wait(bar_mf + cw, (it - 2) & 1);
#pragma unroll
                for (int hf = 0; hf < 2; ++hf) {
                    const int xh = hf * (T::TX / 2) + lane * (VEC / 2);
                    lds_vec<CT, VEC / 2>(mrow + xh, prho[hf]);
                    lds_vec<CT, VEC / 2>(mrow + T::TX + xh, pj[hf][0]);
                    lds_vec<CT, VEC / 2>(mrow + 2 * T::TX + xh, pj[hf][1]);
                    lds_vec<CT, VEC / 2>(mrow + 3 * T::TX + xh, pj[hf][2]);
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(bar_me + cw);
            };
            if constexpr (EARLY) { if (used) take(); }
            // psi of planes it-2, it-1, it (every agent arrives plane by plane, so "it complete" covers the older two)
            mbar_wait(bar_psi + it % NS, (it / NS) & 1);
            if constexpr (!EARLY) { if (used) take(); }
            if (used) {
                const int sc = (it - 1) % NS;
                const unsigned zrow = (unsigned)wrap_m(m0 - 2 + it) * sz + row0;
#pragma unroll
                for (int hf = 0; hf < 2; ++hf) {
                    const int xh = hf * (T::TX / 2) + lane * (VEC / 2);
                    if (xh < txw) {
                        CT S[3][VEC / 2], pc[VEC / 2];
                        psi_sums_rows<L, CT, VEC / 2>(
                            [&](auto DY, auto DZ, auto NX, CT (&t)[VEC / 2], CT& left, CT& right) {
                                const CT* row = psi_row((sc + DZ + NS) % NS, cw + 1 + DY) + T::PAD + xh;
                                lds_vec<CT, VEC / 2>(row, t);
                                if constexpr (NX != 0) { left = row[-1]; right = row[VEC / 2]; }
                            },
                            S, pc);
                        CT A[Q][VEC / 2];
#pragma unroll
                        for (int v = 0; v < VEC / 2; ++v) {
                            const CT rc[1] = {prho[hf][v]}, jc[1][3] = {{pj[hf][0][v], pj[hf][1][v], pj[hf][2][v]}};
                            const CT Sc[1][3] = {{S[0][v], S[1][v], S[2][v]}}, pcc[1] = {pc[v]};
                            CT uc[3], duc[1][3], fc[Q];
                            force_and_velocity<1, CT>(p, rc, jc, Sc, pcc, uc, duc);
                            // tau = 1: f* = f_eq(rho, u' + du) for both forcing schemes (collide() in lbm_hot.cuh, same operations)
                            const CT ub[3] = {uc[0] + duc[0][0], uc[1] + duc[0][1], uc[2] + duc[0][2]};
                            add_feq<L, CT, true>(CT(1), prho[hf][v], ub, fc);
                            static_for<0, Q>([&](auto I) {
                                if constexpr (WREF) A[I][v] = fc[I] - p.wref[I];
                                else A[I][v] = fc[I];
                            });
                        }
                        ST* po = at_u32(static_cast<ST*>(p.f_out), zrow + (unsigned)xh);
                        static_for<0, Q>([&](auto I) { st_vec_global_hint<CT, ST, VEC / 2>(po + (size_t)I * plane, A[I], spol); });
                    }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_free + (it - 2) % NS);   // plane it-2 of the ring has been read for the last time
        }
    };

    // =============================================================== halo rows: up to psi (one landing slot)
    // The landing slot is emptied into registers (rho of the row) as soon as a plane has landed and the copy of the next
    // plane is issued at once, BEFORE this warp waits for room in the psi ring: the copies of the halo rows then run as
    // far ahead as those of the interior rows, i.e. at the time the tile below / above fetches the same rows as its
    // edge rows -- one of the two finds them in L2.
    auto halo_role = [&](int which) {
        const int r = which == 0 ? 0 : nint + 1;
        const int xl = lane * VEC;
        const bool act = xl < txw;
        const RowPipe rp = make_pipe(r);
        ST* slot = halo + (size_t)which * T::RB;
        auto take_rho = [&](int it, CT (&rho)[VEC]) {       // plane it: landing slot -> rho, then refill the slot
            mbar_wait(bar_land + (it & 1) * T::ROWS + r, (it >> 1) & 1);
            CT pair[VEC];
            if (act) {
                const ST* rows = slot + xl;
                static_for<0, Q>([&](auto I) {
                    constexpr int i = I;
                    CT f[VEC];
                    constexpr int so = T::dir_off(i) + T::dir_lead(i);
                    pulled_from_row<CT, ST, VEC, L::E[i][0]>(rows + so, f);
                    if constexpr (WREF) {
#pragma unroll
                        for (int v = 0; v < VEC; ++v) f[v] += p.wref[i];
                    }
                    // rho in the order of density(): f0 + (f1 + f2) + (f3 + f4) + ...
#pragma unroll
                    for (int v = 0; v < VEC; ++v) {
                        if constexpr (i == 0) rho[v] = f[v];
                        else if constexpr (i % 2 == 1) pair[v] = f[v];
                        else rho[v] += pair[v] + f[v];
                    }
                });
            }
            __syncwarp();
            if (it + 1 < nit) issue(rp, r, it + 1, slot);
        };
        issue(rp, r, 0, slot);
        CT rho[VEC], rho_next[VEC];
#pragma unroll
        for (int v = 0; v < VEC; ++v) rho[v] = rho_next[v] = CT(0);
        take_rho(0, rho);
        for (int it = 0; it < nit; ++it) {
            if (it + 1 < nit) take_rho(it + 1, rho_next);
            wait_free(it);
            if (act) {
                CT ps[VEC];
#pragma unroll
                for (int v = 0; v < VEC; ++v) ps[v] = psi_of_rho(p, 0, rho[v]);
                st_vec<CT, CT, VEC>(psi_row(it % NS, r) + T::PAD + xl, ps);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_psi + it % NS);
#pragma unroll
            for (int v = 0; v < VEC; ++v) rho[v] = rho_next[v];
        }
    };

    // =============================================================== ring columns left (side 0) / right (side 1) of the tile
    auto ring_role = [&](int side) {
        const int r = lane;
        const bool act = r <= nint + 1;
        const int xr = side == 0 ? (tx0 > 0 ? tx0 - 1 : p.nx - 1) : (tx0 + txw < p.nx ? tx0 + txw : 0);
        const int xrm = xr > 0 ? xr - 1 : p.nx - 1, xrp1 = xr + 1 < p.nx ? xr + 1 : 0;
        const ST* b[3] = {fin + xrm, fin + xr, fin + xrp1};   // source column for e_x = +1, 0, -1
        const int yw = wrap_y(yb - 1 + r);
        const unsigned yo[3] = {(unsigned)wrap_y(yw - 1) * sy, (unsigned)yw * sy, (unsigned)wrap_y(yw + 1) * sy};
        const int col = side == 0 ? T::PAD - 1 : T::PAD + txw;
        for (int it = 0; it < nit; ++it) {
            const int pl = m0 - 1 + it;
            CT rho = CT(0), pair = CT(0);
            if (act) {
                const unsigned zo[3] = {(unsigned)wrap_m(pl - 1) * sz, (unsigned)wrap_m(pl) * sz, (unsigned)wrap_m(pl + 1) * sz};
                static_for<0, Q>([&](auto I) {
                    constexpr int i = I;
                    constexpr int ex = L::E[i][0], ey = L::E[i][1], ez = L::E[i][2];
                    const unsigned idx = (unsigned)i * plane + zo[1 - ez] + yo[1 - ey];
                    CT f = ld_one<CT, ST>(at_u32(b[1 - ex], idx));
                    if constexpr (WREF) f += p.wref[i];
                    if constexpr (i == 0) rho = f;
                    else if constexpr (i % 2 == 1) pair = f;
                    else rho += pair + f;
                });
            }
            wait_free(it);
            if (act) psi_row(it % NS, r)[col] = psi_of_rho(p, 0, rho);
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_psi + it % NS);
        }
    };

    // role dispatch; whole warpgroups execute setmaxnreg together
    if (warp < T::NCW) {
        reg_inc<T::REG_FRONT>();
        if (warp < TY) front_role();
    } else if (warp < 2 * T::NCW) {
        reg_inc<T::REG_BACK>();
        if (warp - T::NCW < TY) back_role();
    } else {
        reg_dec<T::REG_PROD>();
        const int w = warp - 2 * T::NCW;
        if (w < 2) halo_role(w);
        else ring_role(w - 2);
    }
}

}  // namespace lbmk
