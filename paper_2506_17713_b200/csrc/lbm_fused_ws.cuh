// lbm_fused_ws.cuh -- K2F for D3Q19: the one-pass hot kernel as a warp-specialised producer / consumer pipeline.
//
//   k_fused_ws   S1 (rho, j) + S3 (psi) + S4..S7 in ONE pass over the populations
//                Eq. 4/10, Eq. 12, Eq. 13, Eq. 3, Eq. 5, Eq. 2
//
// A CTA owns an x-y tile of TX x TY cells, marches along z, and recomputes rho -> psi of the one-cell ring around the
// tile from the populations, so that the populations cross HBM once per step (B1 = 2 q s bytes per cell instead of
// B2 = 3 q s + 2 c).  (A first, lock-step version -- every warp loads a plane-row into registers, barrier,
// collide -- was bound by instruction issue and by its phases not overlapping: 5.8 ms on 512^3; removed in round 2.)  Here
// the two halves of the step run concurrently on different planes:
//
//   producers (one warp per tile row incl. the two halo rows, VEC cells per lane, + two warps for the ring columns)
//       plane p: copy the row segments the pull needs (S7 read side: 19 source rows, one per direction, each with one
//       16-byte vector of padding on the side the pull is shifted to in x) from global memory straight into a stage in
//       shared memory with bulk asynchronous copies (cp.async.bulk, SASS UBLKCP; lane i issues direction i; completion
//       on a per-row mbarrier): the whole plane-row is in flight at once and costs no registers.  Then sum rho from
//       the stage, evaluate psi -> psi ring in shared memory.
//   consumers (one warp per interior row)
//       plane m: take the pulled populations from the stage into registers, release the stage, wait for psi of
//       plane m+1, then moments, force from the psi planes m-1, m, m+1, collision, store (S7 write side).
//
//   Hand-over is by mbarriers in shared memory (full / empty per stage, one "psi ready" barrier per ring slot).
//   Producers need few registers, consumers hold Q x VEC values: the register file is re-split with setmaxnreg
//   after the role dispatch.  Earlier versions, measured on 512^3: loads through registers (ptxas split
//   the 29 loads of a plane-row into ~12 batches under the producers' register cap, one memory latency per batch),
//   then per-lane cp.async (LSU-bound issue), then these bulk copies.
//   Addresses are 32-bit element offsets scaled onto per-thread 64-bit bases (mad.wide.u32): two instructions per
//   access instead of five.
// Arithmetic (order of every sum) is that of K1 / K2 in lbm_hot.cuh.
#pragma once
#include "lbm_hot.cuh"

namespace lbmk {

// ------------------------------------------------------------------ mbarrier / register-split primitives (PTX)
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.shared::cta.b64 st, [%0];\n\t}" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n\t.reg .pred p;\n"
        "W%=:\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "\t@p bra D%=;\n\tbra W%=;\n"
        "D%=:\n\t}" ::"r"(smem_u32(bar)), "r"(parity)
        : "memory");
}
template <int N> __device__ __forceinline__ void reg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N)); }
template <int N> __device__ __forceinline__ void reg_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N)); }

// base + idx * sizeof(T) with a 32-bit element index: one IMAD.WIDE.U32
template <class T>
__device__ __forceinline__ const T* at_u32(const T* base, unsigned idx) {
    const T* r;
    asm("mad.wide.u32 %0, %1, %2, %3;" : "=l"(r) : "r"(idx), "n"((int)sizeof(T)), "l"(base));
    return r;
}
template <class T>
__device__ __forceinline__ T* at_u32(T* base, unsigned idx) {
    T* r;
    asm("mad.wide.u32 %0, %1, %2, %3;" : "=l"(r) : "r"(idx), "n"((int)sizeof(T)), "l"(base));
    return r;
}

// bulk asynchronous copy (TMA unit, SASS UBLKCP): `bytes` contiguous bytes global -> shared, 16-byte aligned on both
// sides, completion counted on an mbarrier (complete_tx)
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.expect_tx.shared::cta.b64 st, [%0], %1;\n\t}" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* smem_dst, const void* gmem_src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(smem_dst)),
                 "l"(gmem_src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// TY interior rows per tile, NSTG stages.  With two stages producer and consumer stay coupled (the consumer of plane m
// needs psi of plane m+1, whose copies could only start when the slot of plane m-1 was released): the step period is
// about the mean of their times, not the maximum.  More stages let the copies run AHEAD, but only fit smaller tiles.
template <class L, int NC, class CT, class ST, int VEC, int TY, int NSTG>
struct WsTile {
    static_assert(L::D == 3, "the warp-specialised kernel marches along z");
    static_assert(NSTG >= 2 && NSTG <= 4, "two to four stages");
    static constexpr int AHEAD = NSTG - 2;                         // planes whose copies fly ahead of the one being summed
    static constexpr int Q = L::Q;
    static constexpr int ROWS = TY + 2;
    static constexpr int TX = 32 * VEC;
    static constexpr int PAD = 16 / (int)sizeof(CT);               // psi rows: cells left / right of the tile
    static constexpr int PITCH = TX + 2 * PAD;
    static constexpr int PADS = 16 / (int)sizeof(ST);              // stage rows: one 16-byte vector left / right
    // a staged direction row holds the TX cells of the tile row plus one 16-byte vector on the side its pull is
    // shifted to (left for e_x = +1, right for e_x = -1)
    static constexpr int dir_pitch(int i) { return TX + (L::E[i][0] != 0 ? PADS : 0); }
    static constexpr int dir_lead(int i) { return L::E[i][0] > 0 ? PADS : 0; }          // offset of the tile's first cell
    static constexpr int dir_off(int i) { int o = 0; for (int j = 0; j < i; ++j) o += dir_pitch(j); return o; }
    static constexpr int RB = dir_off(Q);                                                 // one component of a tile row
    static constexpr int NS = NSTG + 3;                            // psi ring slots (>= NSTG + 2, see the hand-over notes)
    // warps come in warpgroups of four (setmaxnreg): consumer group = TY row consumers (+ the two ring warps if two
    // warps are spare there), producer group = ROWS row producers (+ the ring warps otherwise)
    static constexpr int NCONS = TY;                               // row consumers
    static constexpr int NCW = (TY + 3) / 4 * 4;                   // warps of the consumer group
    static constexpr bool RING_IN_CONS = NCW - TY >= 2;
    static constexpr int RING0 = RING_IN_CONS ? TY : NCW + ROWS;   // first ring warp
    static constexpr int NPW = (ROWS + (RING_IN_CONS ? 0 : 2) + 3) / 4 * 4;   // warps of the producer group
    static constexpr int NPSI = ROWS + 2;                          // arrivals per psi plane: row producers + ring warps
    static constexpr int THREADS = (NCW + NPW) * 32;
    static constexpr size_t ROW_ELEMS = (size_t)NC * RB;                            // one tile row, all directions
    static constexpr size_t STAGE_ELEMS = ROW_ELEMS * TY;                           // one stage (interior rows)
    static constexpr size_t PSI_ELEMS = (size_t)NS * NC * ROWS * PITCH;
    static constexpr size_t SMEM = sizeof(ST) * (NSTG * STAGE_ELEMS + 2 * NSTG * ROW_ELEMS) + sizeof(CT) * PSI_ELEMS + 8 * (2 * NSTG + NS + NSTG * ROWS);
    // register split: the pool is THREADS x (registers at launch)
    static constexpr int REG_LAUNCH = (65536 / THREADS) / 8 * 8;
#ifndef LBM_WS_REG_PROD
#define LBM_WS_REG_PROD 56
#endif
    static constexpr int REG_PROD = LBM_WS_REG_PROD;
    static constexpr int REG_CONS_ = ((REG_LAUNCH * THREADS - REG_PROD * NPW * 32) / (NCW * 32)) / 8 * 8;
    static constexpr int REG_CONS = REG_CONS_ > 208 ? 208 : REG_CONS_;
    static_assert(SMEM <= 227 * 1024, "tile does not fit shared memory");
    static_assert(ROWS <= 32, "ring warps map one lane to one row");
    static_assert((VEC * sizeof(ST)) % 4 == 0 && VEC * sizeof(ST) <= 16, "per-lane copy size");
};

// One pulled vector from a staged row: f[v] = row_i[x_v - e_x] for the thread's VEC cells (row points at the lane's
// first cell; the pads hold the neighbouring vectors of the tile edges)
template <class CT, class ST, int VEC, int EX>
__device__ __forceinline__ void pulled_from_row(const ST* row, CT (&f)[VEC]) {
    using R = typename RawVec<sizeof(ST) * VEC>::type;
    const R raw = *reinterpret_cast<const R*>(row);
    const ST* tv = reinterpret_cast<const ST*>(&raw);
    if constexpr (EX == 0) {
#pragma unroll
        for (int v = 0; v < VEC; ++v) f[v] = Cvt<CT, ST>::up(tv[v]);
    } else if constexpr (EX > 0) {
        f[0] = Cvt<CT, ST>::up(row[-1]);
#pragma unroll
        for (int v = 1; v < VEC; ++v) f[v] = Cvt<CT, ST>::up(tv[v - 1]);
    } else {
#pragma unroll
        for (int v = 0; v < VEC - 1; ++v) f[v] = Cvt<CT, ST>::up(tv[v + 1]);
        f[VEC - 1] = Cvt<CT, ST>::up(row[VEC]);
    }
}

template <class L, int NC, class CT, class ST, int COLL, int VEC, int TY, int NSTG, bool WREF>
__global__ void __launch_bounds__((WsTile<L, NC, CT, ST, VEC, TY, NSTG>::THREADS), 1)
k_fused_ws(const __grid_constant__ KParams<CT> p, int mchunk) {
    using T = WsTile<L, NC, CT, ST, VEC, TY, NSTG>;
    constexpr int Q = L::Q;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    ST* stage = reinterpret_cast<ST*>(smem_raw);                        // [NSTG][TY][NC][RB]
    ST* halo = stage + NSTG * T::STAGE_ELEMS;                            // [NSTG planes][2 halo rows][NC][RB] landing rows
    CT* psi_s = reinterpret_cast<CT*>(halo + 2 * NSTG * T::ROW_ELEMS);         // [NS][NC][ROWS][PITCH]
    uint64_t* bars = reinterpret_cast<uint64_t*>(psi_s + T::PSI_ELEMS); // full[NSTG], empty[NSTG], psi_ready[NS]
    uint64_t* bar_full = bars;
    uint64_t* bar_empty = bars + NSTG;
    uint64_t* bar_psi = bars + 2 * NSTG;
    uint64_t* bar_land = bar_psi + T::NS;                               // [NSTG][ROWS] bulk copies of a row producer landed

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int s = 0; s < NSTG; ++s) { mbar_init(bar_full + s, TY); mbar_init(bar_empty + s, T::NCONS); }
        for (int s = 0; s < T::NS; ++s) mbar_init(bar_psi + s, T::NPSI);
        for (int s = 0; s < NSTG * T::ROWS; ++s) mbar_init(bar_land + s, 1);
    }
    __syncthreads();

    const int tx0 = blockIdx.x * T::TX;
    const int txw = min(T::TX, p.nx - tx0);
    const int yb = blockIdx.y * TY;
    const int nint = min(TY, p.ny - yb);                 // interior rows of this tile
    const int nm = p.nz;
    const unsigned sy = (unsigned)p.nx, sz = (unsigned)p.nx * (unsigned)p.ny;
    const int m0 = blockIdx.z * mchunk, m1 = min(nm, m0 + mchunk);
    const unsigned plane = (unsigned)p.plane;
    auto wrap_y = [&](int y) { return y < 0 ? y + p.ny : (y >= p.ny ? y - p.ny : y); };
    auto wrap_m = [&](int m) { return m < 0 ? m + nm : (m >= nm ? m - nm : m); };
    auto psi_row = [&](int slot, int k, int r) { return psi_s + ((size_t)(slot * NC + k) * T::ROWS + r) * T::PITCH; };

    const ST* fin = static_cast<const ST*>(p.f_in);

    // ---- ring role: the columns left (side 0) / right (side 1) of the tile, one lane per tile row
    auto ring_role = [&](int side) {
        const int r = lane;
        const bool act = r <= nint + 1;
        const int xr = side == 0 ? (tx0 > 0 ? tx0 - 1 : p.nx - 1) : (tx0 + txw < p.nx ? tx0 + txw : 0);
        const int xrm = xr > 0 ? xr - 1 : p.nx - 1, xrp = xr + 1 < p.nx ? xr + 1 : 0;
        const ST* b[3] = {fin + xrm, fin + xr, fin + xrp};   // source column for e_x = +1, 0, -1
        const int yw = wrap_y(yb - 1 + r);
        const unsigned yo[3] = {(unsigned)wrap_y(yw - 1) * sy, (unsigned)yw * sy, (unsigned)wrap_y(yw + 1) * sy};
        const int col = side == 0 ? T::PAD - 1 : T::PAD + txw;
        for (int pl = m0 - 1; pl <= m1; ++pl) {
            const int it = pl - m0;
            if (it >= 0) mbar_wait(bar_empty + it % NSTG, ((it / NSTG) & 1) ^ 1);   // pacing only
            const int q = it + 1, slot = q % T::NS;
            if (act) {
                const unsigned zo[3] = {(unsigned)wrap_m(pl - 1) * sz, (unsigned)wrap_m(pl) * sz, (unsigned)wrap_m(pl + 1) * sz};
#pragma unroll
                for (int k = 0; k < NC; ++k) {
                    CT rho = CT(0), pair = CT(0);
                    static_for<0, Q>([&](auto I) {
                        constexpr int i = I;
                        constexpr int ex = L::E[i][0], ey = L::E[i][1], ez = L::E[i][2];
                        const unsigned idx = (unsigned)(k * Q + i) * plane + zo[1 - ez] + yo[1 - ey];
                        CT f = ld_one<CT, ST>(at_u32(b[1 - ex], idx));
                        if constexpr (WREF) f += p.wref[i];
                        if constexpr (i == 0) rho = f;
                        else if constexpr (i % 2 == 1) pair = f;
                        else rho += pair + f;
                    });
                    psi_row(slot, k, r)[col] = psi_of_rho(p, k, rho);
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_psi + slot);
        }
    };

    // =============================================================== consumers
    auto consumer_role = [&]() {
        const int cw = warp;               // interior row index 0..TY-1  (tile row r = cw + 1)
        const int xl = lane * VEC;
        const bool act = cw < nint && xl < txw;
        const int yw = wrap_y(yb + cw);
        const unsigned cell0 = (unsigned)yw * sy + (unsigned)(tx0 + xl);
        for (int m = m0; m < m1; ++m) {
            const int it = m - m0, s = it % NSTG;
            mbar_wait(bar_full + s, (it / NSTG) & 1);
            CT A[NC][Q][VEC];
            if (act) {
                const ST* rows = stage + (size_t)s * T::STAGE_ELEMS + (size_t)cw * T::ROW_ELEMS + xl;
#pragma unroll
                for (int k = 0; k < NC; ++k)
                    static_for<0, Q>([&](auto I) {
                        constexpr int i = I;
                        // layout constants forced to compile-time values (evaluated at run time they would read the host-side
                        // lattice table: the compiler then treats the path as unreachable and silently drops it)
                        constexpr int so = T::dir_off(i) + T::dir_lead(i);
                        pulled_from_row<CT, ST, VEC, L::E[i][0]>(rows + k * T::RB + so, A[k][i]);
                    });
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_empty + s);
            // psi of planes m-1, m, m+1: plane q (counted from m0-1) lives in slot q % NS
            const int qn = it + 2;
            mbar_wait(bar_psi + (qn % T::NS), (qn / T::NS) & 1);
            if (!act) continue;
            const int sc = (it + 1) % T::NS;
            CT S[NC][3][VEC], pc[NC][VEC];
            if constexpr (COLL != 2) {
#pragma unroll
                for (int kp = 0; kp < NC; ++kp) {
                    psi_sums_rows<L, CT, VEC>(
                        [&](auto DY, auto DZ, auto NX, CT (&t)[VEC], CT& left, CT& right) {
                            const CT* row = psi_row((sc + DZ + T::NS) % T::NS, kp, cw + 1 + DY) + T::PAD + xl;
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
#pragma unroll
            for (int v = 0; v < VEC; ++v) {
                CT fc[NC][Q];
#pragma unroll
                for (int k = 0; k < NC; ++k)
                    static_for<0, Q>([&](auto I) {
                        if constexpr (WREF) fc[k][I] = A[k][I][v] + p.wref[I];
                        else fc[k][I] = A[k][I][v];
                    });
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
                for (int k = 0; k < NC; ++k)
                    static_for<0, Q>([&](auto I) {
                        if constexpr (WREF) A[k][I][v] = fc[k][I] - p.wref[I];
                        else A[k][I][v] = fc[k][I];
                    });
            }
            ST* po = at_u32(static_cast<ST*>(p.f_out), (unsigned)wrap_m(m) * sz + cell0);
#pragma unroll
            for (int k = 0; k < NC; ++k)
                static_for<0, Q>([&](auto I) {
                    st_vec_global<CT, ST, VEC>(po + (size_t)(k * Q + I) * plane, A[k][I]);
                });
        }
    };
    // =============================================================== producers
    auto producer_role = [&](int r) {
        {
            // ---- row producer: tile row r (0 and nint+1 are the halo rows)
            const int xl = lane * VEC;
            const bool used = r <= nint + 1;
            const bool act = used && xl < txw;
            const bool interior = r >= 1 && r <= nint;
            const int yw = wrap_y(yb - 1 + r);
            // the 16-byte vectors just left / right of the tile (periodic wrap), copied by lane 0 / the last lane
            const int xlp = (tx0 > 0 ? tx0 : p.nx) - T::PADS;
            const int xrp = tx0 + txw < p.nx ? tx0 + txw : 0;
            // lane i < Q issues the bulk copies of direction i: source row (y - e_y, z - e_z) of its plane
            int ex_l = 0, ey_l = 0, ez_l = 0, off_l = 0;
            static_for<0, Q>([&](auto I) {
                constexpr int ex = L::E[I][0], ey = L::E[I][1], ez = L::E[I][2], so = T::dir_off(I);
                if (lane == I) { ex_l = ex; ey_l = ey; ez_l = ez; off_l = so; }
            });
            const unsigned base_l = (unsigned)lane * plane + (unsigned)wrap_y(yw - ey_l) * sy;
            constexpr int NXD = []() { int n = 0; for (int i = 0; i < Q; ++i) n += L::E[i][0] != 0; return n; }();
            const uint32_t main_bytes = (uint32_t)txw * (uint32_t)sizeof(ST);
            const uint32_t land_bytes = (uint32_t)NC * ((uint32_t)Q * main_bytes + (uint32_t)NXD * 16u);
            // where plane pl of this row lands: interior rows in stage (it mod NSTG), halo rows in their own two buffers
            auto landing = [&](int it) -> ST* {
                return interior ? stage + (size_t)((it + NSTG) % NSTG) * T::STAGE_ELEMS + (size_t)(r - 1) * T::ROW_ELEMS
                                : halo + (size_t)(2 * ((it + NSTG) % NSTG) + (r == 0 ? 0 : 1)) * T::ROW_ELEMS;
            };
            // start the copies of plane pl (after its stage slot has been released by the consumers)
            auto issue = [&](int pl) {
                const int it = pl - m0;
                if (it >= 0) mbar_wait(bar_empty + it % NSTG, ((it / NSTG) & 1) ^ 1);
                if (!used) return;
                uint64_t* lb = bar_land + ((it + NSTG) % NSTG) * T::ROWS + r;
                ST* land = landing(it);
                if (lane == 0) mbar_expect_tx(lb, land_bytes);
                __syncwarp();
                if (lane < Q) {
                    const unsigned idx0 = base_l + (unsigned)wrap_m(pl - ez_l) * sz;
#pragma unroll
                    for (int k = 0; k < NC; ++k) {
                        const ST* src = fin + ((size_t)k * Q * plane + idx0);
                        ST* dst = land + k * T::RB + off_l;
                        // the pad vector is contiguous with the row segment unless the tile touches the periodic seam
                        if (ex_l > 0) {
                            if (tx0 > 0) bulk_g2s(dst, src + (tx0 - T::PADS), main_bytes + 16u, lb);
                            else { bulk_g2s(dst + T::PADS, src + tx0, main_bytes, lb); bulk_g2s(dst, src + xlp, 16u, lb); }
                        } else if (ex_l < 0) {
                            if (tx0 + txw < p.nx) bulk_g2s(dst, src + tx0, main_bytes + 16u, lb);
                            else { bulk_g2s(dst, src + tx0, main_bytes, lb); bulk_g2s(dst + txw, src + xrp, 16u, lb); }
                        } else {
                            bulk_g2s(dst, src + tx0, main_bytes, lb);
                        }
                    }
                }
            };
            // With more than two stages the copies run AHEAD planes in front of the plane being summed, so that the
            // memory system always has a plane in flight.  (With two stages that does not work: the slot of plane pl+1 is
            // only released once the consumers have collided plane pl-2, and the producer would block in front of a rho
            // pass whose data has already landed.)
#pragma unroll
            for (int d = 0; d < T::AHEAD; ++d)
                if (m0 - 1 + d <= m1) issue(m0 - 1 + d);
            for (int pl = m0 - 1; pl <= m1; ++pl) {
                const int it = pl - m0;                       // -1 .. mchunk
                const bool staged = it >= 0 && pl < m1;       // planes m0-1 and m1 only feed psi
                const int s = (it + NSTG) % NSTG;
                if (pl + T::AHEAD <= m1) issue(pl + T::AHEAD);
                const int q = it + 1, slot = q % T::NS;
                const ST* land = landing(it);
                if (used) mbar_wait(bar_land + s * T::ROWS + r, ((it + 1) / NSTG) & 1);
                if (act) {
#pragma unroll
                    for (int k = 0; k < NC; ++k) {
                        CT rho[VEC], pair[VEC];
                        static_for<0, Q>([&](auto I) {
                            constexpr int i = I;
                            CT f[VEC];
                            constexpr int so = T::dir_off(i) + T::dir_lead(i);
                            pulled_from_row<CT, ST, VEC, L::E[i][0]>(land + k * T::RB + so + xl, f);
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
                        CT ps[VEC];
#pragma unroll
                        for (int v = 0; v < VEC; ++v) ps[v] = psi_of_rho(p, k, rho[v]);
                        st_vec<CT, CT, VEC>(psi_row(slot, k, r) + T::PAD + xl, ps);
                    }
                }
                __syncwarp();
                if (lane == 0) {
                    mbar_arrive(bar_psi + slot);
                    if (staged && r >= 1 && r <= TY) mbar_arrive(bar_full + s);
                }
            }
        }
    };

    // role dispatch; whole warpgroups execute setmaxnreg together
    if (warp < T::NCW) {
        reg_inc<T::REG_CONS>();
        if (warp < T::NCONS) consumer_role();
        else if (T::RING_IN_CONS && warp >= T::RING0 && warp < T::RING0 + 2) ring_role(warp - T::RING0);
    } else {
        reg_dec<T::REG_PROD>();
        if (warp < T::NCW + T::ROWS) producer_role(warp - T::NCW);
        else if (!T::RING_IN_CONS && warp >= T::RING0 && warp < T::RING0 + 2) ring_role(warp - T::RING0);
    }
}

}  // namespace lbmk
