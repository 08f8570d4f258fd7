// lbm_fused_eq.cuh -- K2F for D3Q19 when the post-collision state is an equilibrium: row pipelines.
//
//   k_fused_eq   S1 (rho, j) + S3 (psi) + S4..S7 in ONE pass over the populations, for one component, BGK with tau = 1
//                (both forcing schemes then give f* = f_eq(rho, u' + F/rho): Eq. 3 + Eq. 5; R7) -- configs 5
//                and the paper's own benchmark case.
//
// What bounds k_fused_ws (lbm_fused_ws.cuh) is the coupling of its two stages: the consumer of plane m needs psi of plane
// m+1, which the producers can only sum after the copies of plane m+1 have landed, and those could only start once the
// consumers had emptied a slot.  Here the collision needs nothing of a plane but its moments, so the dependency is cut
// at the registers instead:
//
//   consumer warp of tile row r, plane pl:
//       wait for ITS row of plane pl to land in ITS slot of the stage (bulk asynchronous copies, one mbarrier per row and
//       slot) -> registers -> rho, j (S1) -> the slot is free again: the same warp issues the copies of plane pl+2 into
//       it (no hand-over to a producer, no barrier between warps) -> psi(rho) to the psi ring -> wait until the ring
//       holds plane pl completely -> force, f_eq(rho, u' + du) and store of the PENDING plane pl-1, of which only
//       rho and j (16 registers) were kept.
//   two halo-row warps do the same for the rows above / below the tile up to psi (their rows are never collided),
//   two ring warps the columns left / right of it with scalar loads.
//
// Every row is its own two-slot pipeline; the warps meet only at the psi ring (one "plane complete" mbarrier per ring
// slot, one "slot free" mbarrier for the halo / ring warps that run ahead).  The copies of plane pl+2 are in flight while
// plane pl-1 is collided and plane pl+1 waits in the other slot.
// CPS = 1: tiles of 32 x VEC cells by TY rows, one CTA per SM; CPS = 2: half-width tiles (VEC / 2 cells per lane), two CTAs
// per SM -- chosen for rows that leave much of a full-width tile idle (416 = 3.25 x 128) and for domains with few tiles.
// Measured on C5-512 and kept out: bulk copies issued by dedicated copy warps (same time: the consumers are
// not issue-bound), one 4-D tensor-map box per direction instead of 190 row copies with either a TMA-stored staging
// area (room for one landing slot only: 4.8 ms) or two landing slots (5.1 ms), the stores of a plane issued after the
// shared-memory loads of the next (4.3 ms), stores per cell pair (half sectors: 5.1 ms).  What is left, from the stall
// samples: the eight rows collide and store in the same phase, the 78 KB burst drains at ~40 B/cycle while the arithmetic
// pipes idle (copies alone 1.9 ms, + arithmetic 2.9 ms, + stores 3.9 ms).
// Arithmetic (order of every sum) is that of K1 / K2 in lbm_hot.cuh: results are bit-identical to the two-pass path.
#pragma once
#include "lbm_fused_ws.cuh"

namespace lbmk {

template <class L, class CT, class ST, int VEC, int TY, int CPS>
struct EqTile {
    static_assert(L::D == 3, "the kernel marches along z");
    static constexpr int Q = L::Q;
    static constexpr int NSTG = 2;                                  // slots per row
    static constexpr int NS = 4;                                    // psi ring slots (see the hand-over notes in the kernel)
    static constexpr int ROWS = TY + 2;
    static constexpr int TX = 32 * VEC;
    static constexpr int PAD = 16 / (int)sizeof(CT);                // psi rows: cells left / right of the tile
    static constexpr int PITCH = TX + 2 * PAD;
    static constexpr int PADS = 16 / (int)sizeof(ST);               // stage rows: one 16-byte vector left / right
    static constexpr int dir_pitch(int i) { return TX + (L::E[i][0] != 0 ? PADS : 0); }
    static constexpr int dir_lead(int i) { return L::E[i][0] > 0 ? PADS : 0; }
    static constexpr int dir_off(int i) { int o = 0; for (int j = 0; j < i; ++j) o += dir_pitch(j); return o; }
    static constexpr int RB = dir_off(Q);                           // one tile row, all directions
    static constexpr int NCW = (TY + 3) / 4 * 4;                    // warps of the consumer group (TY row consumers)
    static constexpr int NPW = 4;                                   // producer group: two halo rows, two ring columns
    static constexpr int NPSI = TY + 4;                             // arrivals per psi plane
    static constexpr int THREADS = (NCW + NPW) * 32;
    static constexpr size_t STAGE_ELEMS = (size_t)RB * TY;
    static constexpr size_t PSI_ELEMS = (size_t)NS * ROWS * PITCH;
    static constexpr int NBAR = NSTG * ROWS + 2 * NS;
    static constexpr size_t SMEM = sizeof(ST) * (NSTG * STAGE_ELEMS + 2 * NSTG * (size_t)RB) + sizeof(CT) * PSI_ELEMS + 8 * NBAR;
    // register split (setmaxnreg): the pool is THREADS x (registers at launch)
    static constexpr int REG_LAUNCH = (65536 / CPS / THREADS) / 8 * 8;
    static constexpr int REG_PROD = CPS == 1 ? 56 : 40;
    static constexpr int REG_CONS_ = ((REG_LAUNCH * THREADS - REG_PROD * NPW * 32) / (NCW * 32)) / 8 * 8;
    static constexpr int REG_CONS = REG_CONS_ > 232 ? 232 : REG_CONS_;
    static_assert(SMEM <= (CPS == 1 ? 227 : 113) * 1024, "tile does not fit shared memory");
    static_assert(ROWS <= 32, "ring warps map one lane to one row");
};

template <class L, class CT, class ST, int VEC, int TY, int CPS, bool WREF>
__global__ void __launch_bounds__((EqTile<L, CT, ST, VEC, TY, CPS>::THREADS), CPS)
k_fused_eq(const __grid_constant__ KParams<CT> p, int mchunk) {
    using T = EqTile<L, CT, ST, VEC, TY, CPS>;
    constexpr int Q = L::Q, NSTG = T::NSTG, NS = T::NS;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    ST* stage = reinterpret_cast<ST*>(smem_raw);                          // [NSTG][TY][RB]
    ST* halo = stage + NSTG * T::STAGE_ELEMS;                              // [NSTG][2][RB]
    CT* psi_s = reinterpret_cast<CT*>(halo + 2 * NSTG * T::RB);            // [NS][ROWS][PITCH]
    uint64_t* bar_land = reinterpret_cast<uint64_t*>(psi_s + T::PSI_ELEMS);   // [NSTG][ROWS] copies of a row landed
    uint64_t* bar_psi = bar_land + NSTG * T::ROWS;                         // [NS] psi of a plane complete
    uint64_t* bar_free = bar_psi + NS;                                     // [NS] ring slot read for the last time

    const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);   // uniform, and known to be so
    const int lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int s = 0; s < NSTG * T::ROWS; ++s) mbar_init(bar_land + s, 1);
        for (int s = 0; s < NS; ++s) { mbar_init(bar_psi + s, T::NPSI); mbar_init(bar_free + s, TY); }
    }
    __syncthreads();

    const int tx0 = blockIdx.x * T::TX;
    const int txw = min(T::TX, p.nx - tx0);
    const int yb = blockIdx.y * TY;
    const int nint = min(TY, p.ny - yb);                  // interior rows of this tile
    const int nm = p.nz;
    const unsigned sy = (unsigned)p.nx, sz = (unsigned)p.nx * (unsigned)p.ny;
    const int m0 = blockIdx.z * mchunk, m1 = min(nm, m0 + mchunk);
    const int nit = m1 - m0 + 2;                          // planes m0-1 .. m1 pass through the pipeline (it = 0 .. nit-1)
    const unsigned plane = (unsigned)p.plane;
    auto wrap_y = [&](int y) { return y < 0 ? y + p.ny : (y >= p.ny ? y - p.ny : y); };
    auto wrap_m = [&](int m) { return m < 0 ? m + nm : (m >= nm ? m - nm : m); };
    auto psi_row = [&](int slot, int r) { return psi_s + ((size_t)slot * T::ROWS + r) * T::PITCH; };
    const ST* fin = static_cast<const ST*>(p.f_in);

    // ---- the row pipeline of consumers and halo warps: tile row r (0 and nint+1 are the halo rows), two landing slots.
    // Lane i < Q issues the bulk copies of direction i (S7 read side: source row y - e_y of plane z - e_z, with one
    // 16-byte vector of padding on the side the pull is shifted to in x).
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
    const int xlp = (tx0 > 0 ? tx0 : p.nx) - T::PADS;      // the 16-byte vectors just left / right of the tile (periodic wrap)
    const int xrp = tx0 + txw < p.nx ? tx0 + txw : 0;
    auto issue = [&](const RowPipe& rp, int r, int it, ST* land) {
        uint64_t* lb = bar_land + (it & 1) * T::ROWS + r;
        if (lane == 0) mbar_expect_tx(lb, land_bytes);
        __syncwarp();
        if (lane < Q) {
            const int pl = m0 - 1 + it;
            const ST* src = fin + (rp.base_l + (unsigned)wrap_m(pl - rp.ez_l) * sz);
            ST* dst = land + rp.off_l;
            // the pad vector is contiguous with the row segment unless the tile touches the periodic seam
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

    // =============================================================== consumers: one warp per interior row
    auto consumer_role = [&]() {
        const int cw = warp, r = cw + 1;
        const int xl = lane * VEC;
        const bool used = cw < nint;
        const bool act = used && xl < txw;
        const unsigned cell0 = (unsigned)wrap_y(yb + cw) * sy + (unsigned)(tx0 + xl);
        auto slot_of = [&](int it) { return stage + (size_t)(it & 1) * T::STAGE_ELEMS + (size_t)cw * T::RB; };
        const RowPipe rp = make_pipe(r);
        if (used) {
            issue(rp, r, 0, slot_of(0));
            issue(rp, r, 1, slot_of(1));
        }
        // pulled populations of plane it: shared memory -> registers
        auto load_plane = [&](int it, CT (&A)[Q][VEC]) {
            const ST* rows = slot_of(it) + xl;
            static_for<0, Q>([&](auto I) {
                constexpr int i = I;
                constexpr int so = T::dir_off(i) + T::dir_lead(i);   // compile-time (see lbm_fused_ws.cuh)
                pulled_from_row<CT, ST, VEC, L::E[i][0]>(rows + so, A[i]);
            });
        };
        auto moments_of = [&](const CT (&A)[Q][VEC], CT (&rho)[VEC], CT (&j)[3][VEC]) {
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
        };
        CT prho[VEC], pj[3][VEC];                          // the pending plane it-1: its moments
        for (int it = 0; it < nit; ++it) {
            CT rho[VEC], j[3][VEC];
            if (used) mbar_wait(bar_land + (it & 1) * T::ROWS + r, (it >> 1) & 1);
            if (act) {
                CT A[Q][VEC];
                load_plane(it, A);
                moments_of(A, rho, j);
            }
            __syncwarp();                                   // every lane has its values: the slot can be overwritten
            if (used && it + 2 < nit) issue(rp, r, it + 2, slot_of(it));
            const int slot = it % NS;
            if (act) {
                CT ps[VEC];
#pragma unroll
                for (int v = 0; v < VEC; ++v) ps[v] = psi_of_rho(p, 0, rho[v]);
                st_vec<CT, CT, VEC>(psi_row(slot, r) + T::PAD + xl, ps);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_psi + slot);
            if (it >= 2) {
                // psi of planes it-2, it-1, it (every agent arrives plane by plane, so "it complete" covers the older two).
                // Writing plane it into the slot of plane it-NS above needed no wait: to be here a warp has passed this wait
                // for plane it-1, i.e. every consumer had arrived for it-1 and so had finished its reads of plane it-NS = it-4
                // (last needed by the collision of pending plane it-3).
                mbar_wait(bar_psi + slot, (it / NS) & 1);
                if (act) {
                    const int sc = (it - 1) % NS;
                    CT S[3][VEC], pc[VEC];
                    psi_sums_rows<L, CT, VEC>(
                        [&](auto DY, auto DZ, auto NX, CT (&t)[VEC], CT& left, CT& right) {
                            const CT* row = psi_row((sc + DZ + NS) % NS, cw + 1 + DY) + T::PAD + xl;
                            using R = typename RawVec<sizeof(CT) * VEC>::type;
                            const R raw = *reinterpret_cast<const R*>(row);
                            const CT* tv = reinterpret_cast<const CT*>(&raw);
#pragma unroll
                            for (int v = 0; v < VEC; ++v) t[v] = tv[v];
                            if constexpr (NX != 0) { left = row[-1]; right = row[VEC]; }
                        },
                        S, pc);
                    CT A[Q][VEC];
#pragma unroll
                    for (int v = 0; v < VEC; ++v) {
                        const CT rc[1] = {prho[v]}, jc[1][3] = {{pj[0][v], pj[1][v], pj[2][v]}};
                        const CT Sc[1][3] = {{S[0][v], S[1][v], S[2][v]}}, pcc[1] = {pc[v]};
                        CT uc[3], duc[1][3], fc[Q];
                        force_and_velocity<1, CT>(p, rc, jc, Sc, pcc, uc, duc);
                        // tau = 1: f* = f_eq(rho, u' + du) for both forcing schemes (collide() in lbm_hot.cuh, same operations)
                        const CT ub[3] = {uc[0] + duc[0][0], uc[1] + duc[0][1], uc[2] + duc[0][2]};
                        add_feq<L, CT, true>(CT(1), prho[v], ub, fc);
                        static_for<0, Q>([&](auto I) {
                            if constexpr (WREF) A[I][v] = fc[I] - p.wref[I];
                            else A[I][v] = fc[I];
                        });
                    }
                    ST* po = at_u32(static_cast<ST*>(p.f_out), (unsigned)wrap_m(m0 - 2 + it) * sz + cell0);
                    static_for<0, Q>([&](auto I) { st_vec_global<CT, ST, VEC>(po + (size_t)I * plane, A[I]); });
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(bar_free + (it - 2) % NS);   // plane it-2 of the ring has been read for the last time
            }
#pragma unroll
            for (int v = 0; v < VEC; ++v) { prho[v] = rho[v]; pj[0][v] = j[0][v]; pj[1][v] = j[1][v]; pj[2][v] = j[2][v]; }
        }
    };

    // a ring slot is rewritten with plane `it` once the consumers have read plane it-NS for the last time
    auto wait_free = [&](int it) {
        if (it >= NS) mbar_wait(bar_free + it % NS, (it / NS - 1) & 1);
    };

    // =============================================================== halo rows: up to psi
    auto halo_role = [&](int which) {
        const int r = which == 0 ? 0 : nint + 1;
        const int xl = lane * VEC;
        const bool act = xl < txw;
        const RowPipe rp = make_pipe(r);
        auto slot_of = [&](int it) { return halo + (size_t)(2 * (it & 1) + which) * T::RB; };
        issue(rp, r, 0, slot_of(0));
        issue(rp, r, 1, slot_of(1));
        for (int it = 0; it < nit; ++it) {
            mbar_wait(bar_land + (it & 1) * T::ROWS + r, (it >> 1) & 1);
            CT rho[VEC], pair[VEC];
            if (act) {
                const ST* rows = slot_of(it) + xl;
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
            if (it + 2 < nit) issue(rp, r, it + 2, slot_of(it));
            wait_free(it);
            if (act) {
                CT ps[VEC];
#pragma unroll
                for (int v = 0; v < VEC; ++v) ps[v] = psi_of_rho(p, 0, rho[v]);
                st_vec<CT, CT, VEC>(psi_row(it % NS, r) + T::PAD + xl, ps);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_psi + it % NS);
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
        reg_inc<T::REG_CONS>();
        if (warp < TY) consumer_role();
    } else {
        reg_dec<T::REG_PROD>();
        const int w = warp - T::NCW;
        if (w < 2) halo_role(w);
        else ring_role(w - 2);
    }
}

}  // namespace lbmk
