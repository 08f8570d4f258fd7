// lbm_small.cuh -- the step of small, launch-bound domains as ONE persistent kernel for n time steps.
//
//   k_steps_tile   (2-D lattices; configs 1 and 2)  n x [ A: rho, psi on the CTA's tile and a ring around it | B: virtual
//                  density in shared memory | C: stream, force, collide, boundaries | grid barrier ]   -- below
//   k_steps_coop   (any lattice)  n x [ K1: rho, psi  |  grid barrier  |  K1b: virtual density  |  grid barrier  |  K2: stream,
//                  force, collide, boundaries  |  grid barrier ]          (S1..S7; citations as in lbm_hot.cuh)
//
// Configs 1 and 2 (0.3 MB and 9.4 MB of state) live in L2 and a step is two or three kernels of a few microseconds: what
// a step costs there is the launch and drain of each kernel, even when replayed from a CUDA graph with programmatic
// dependent launches (11.5 us per step on config 2, 5 us on config 1).  Here the CTAs stay resident (cooperative launch),
// keep their cells for all n steps, and meet at a grid barrier between the phases: one atomic per CTA on a monotonic
// counter, polled with acquire loads.  Everything a phase reads was written by other SMs in the phase before, so global
// data is loaded with ld.global.cg (L2 only; the read-only path of the other kernels could serve stale L1 lines).
// k_steps_coop is used where every cell gets its own resident thread (config 1: 4.8 -> 4.3 us per step; on config 2, where a
// thread would take two cells in turn, it loses to the separate vectorised kernels under graph replay: 14.2 against 11.3 us);
// k_steps_tile needs ONE barrier per step (config 1: 2.2 us, config 2: 6.4 us) and is what lbm_step picks on 2-D lattices.
// One cell per thread; the arithmetic is that of k_moments_v / k_virtual_density / k_step_v (same device functions, same
// order of every sum), so the result is bit-identical to the plain launches (tested).
#pragma once
#include "lbm_hot.cuh"

namespace lbmk {

__device__ __forceinline__ void grid_barrier(unsigned* ctr, unsigned& target, unsigned nblocks) {
    __syncthreads();
    target += nblocks;
    if (threadIdx.x == 0) {
        asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(ctr) : "memory");
        unsigned v;
        do {
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(ctr) : "memory");
        } while ((int)(v - target) < 0);
    }
    __syncthreads();
}

template <class CT, class ST> struct CgLoad;
template <> struct CgLoad<float, float> { static __device__ __forceinline__ float ld(const float* p) { return __ldcg(p); } };
template <> struct CgLoad<double, double> { static __device__ __forceinline__ double ld(const double* p) { return __ldcg(p); } };
template <> struct CgLoad<double, float> { static __device__ __forceinline__ double ld(const float* p) { return (double)__ldcg(p); } };
template <> struct CgLoad<float, __half> {
    static __device__ __forceinline__ float ld(const __half* p) {
        return __half2float(__ushort_as_half(__ldcg(reinterpret_cast<const unsigned short*>(p))));
    }
};

// S7 read side (as pull() in lbm_core.cuh, L2 loads)
template <class L, class CT, class ST, bool BND>
__device__ __forceinline__ void pull_cg(const KParams<CT>& p, const ST* fin, const Cell& c, uint32_t fl, int k, CT (&f)[L::Q]) {
    const ST* base = fin + (long long)k * L::Q * p.plane;
    static_for<0, L::Q>([&](auto I) {
        constexpr int i = I;
        constexpr int ib = opposite<L>(i);
        const ST* src = base + (long long)i * p.plane + c.id;
        if constexpr (i > 0) {
            const int off = nbr_offset<-L::E[i][0], -L::E[i][1], -L::E[i][2]>(c);
            if (BND && ((fl >> i) & 1u)) src = base + (long long)ib * p.plane + c.id;
            else src += off;
        }
        f[i] = CgLoad<CT, ST>::ld(src) + p.wref[i];
    });
}

template <class L, int NC, class CT, class ST, int COLL, bool BND>
__global__ void __launch_bounds__(256) k_steps_coop(const __grid_constant__ KParams<CT> p, int nsteps, unsigned* ctr) {
    const ST* fa = static_cast<const ST*>(p.f_in);
    ST* fb = static_cast<ST*>(p.f_out);
    const int gsize = gridDim.x * blockDim.x, gtid = blockIdx.x * blockDim.x + threadIdx.x;
    unsigned target = 0;
    for (int s = 0; s < nsteps; ++s) {
        if constexpr (COLL != 2) {
            // ---- K1: rho, psi at the fluid cells
            for (int id = gtid; id < p.N; id += gsize) {
                uint32_t fl = 0;
                if constexpr (BND) fl = __ldg(p.flags + id);
                if (fl & SOLID_BIT) continue;
                const Cell c = make_cell<L>(p, id);
#pragma unroll
                for (int k = 0; k < NC; ++k) {
                    CT f[L::Q];
                    pull_cg<L, CT, ST, BND>(p, fa, c, fl, k, f);
                    const CT r = density<L, CT>(f);
                    p.psi[(long long)k * p.N + id] = psi_of_rho(p, k, r);
                    if (p.write_rho) p.rho[(long long)k * p.N + id] = r;
                }
            }
            grid_barrier(ctr, target, gridDim.x);
            // ---- K1b: virtual density at the boundary solids (S2, Eq. 17)
            if (p.nbsolid > 0) {
                for (int b = gtid; b < p.nbsolid; b += gsize) {
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
                            for (int k = 0; k < NC; ++k) num[k] += w * __ldcg(p.rho + (long long)k * p.N + nb);
                        }
                    });
#pragma unroll
                    for (int k = 0; k < NC; ++k) {
                        CT rs = p.wet_phi[k] * (num[k] / den) - p.wet_drho[k];
                        rs = rs < p.wet_lo[k] ? p.wet_lo[k] : rs;
                        rs = rs > p.wet_hi[k] ? p.wet_hi[k] : rs;
                        p.rho[(long long)k * p.N + id] = rs;
                        p.psi[(long long)k * p.N + id] = psi_of_rho(p, k, rs);
                    }
                }
                grid_barrier(ctr, target, gridDim.x);
            }
        }
        // ---- K2: stream, moments, force, collide, boundary rules
        for (int id = gtid; id < p.N; id += gsize) {
            uint32_t fl = 0;
            if constexpr (BND) fl = __ldg(p.flags + id);
            if (fl & SOLID_BIT) continue;
            const Cell c = make_cell<L>(p, id);
            CT f[NC][L::Q], rho[NC], j[NC][3];
#pragma unroll
            for (int k = 0; k < NC; ++k) {
                pull_cg<L, CT, ST, BND>(p, fa, c, fl, k, f[k]);
                if constexpr (COLL != 2) moments<L, CT>(f[k], rho[k], j[k]);
            }
            CT u[3] = {CT(0), CT(0), CT(0)}, du[NC][3];
            if constexpr (COLL != 2) {
                CT S[NC][3], pc[NC];
#pragma unroll
                for (int kp = 0; kp < NC; ++kp) {
                    const CT* ps = p.psi + (long long)kp * p.N + id;
                    auto rowfn = [&](auto DY, auto DZ, auto NX, CT (&t)[1], CT& left, CT& right) {
                        constexpr int dy = DY, dz = DZ;
                        t[0] = __ldcg(ps + nbr_offset<0, dy, dz>(c));
                        if constexpr (NX != 0) {
                            left = __ldcg(ps + nbr_offset<-1, dy, dz>(c));
                            right = __ldcg(ps + nbr_offset<1, dy, dz>(c));
                        }
                    };
                    CT S1[3][1], pc1[1];
                    psi_sums_rows<L, CT, 1>(rowfn, S1, pc1);
                    S[kp][0] = S1[0][0]; S[kp][1] = S1[1][0]; S[kp][2] = S1[2][0];
                    pc[kp] = pc1[0];
                }
                force_and_velocity<NC, CT>(p, rho, j, S, pc, u, du);
            }
#pragma unroll
            for (int k = 0; k < NC; ++k) {
                if constexpr (COLL != 2) collide<L, COLL, CT>(p, k, rho[k], u, du[k], f[k]);
                if constexpr (BND) {
                    if (fl & FACEBC_BIT) apply_face_rules<L, CT>(p, c, k, u, f[k]);
                }
                ST* out = fb + (long long)k * L::Q * p.plane + id;
                static_for<0, L::Q>([&](auto I) { Conv<CT, ST>::st(out + (long long)I * p.plane, f[k][I] - p.wref[I]); });
            }
        }
        grid_barrier(ctr, target, gridDim.x);
        const ST* t_ = fa; fa = fb; fb = const_cast<ST*>(t_);
    }
}

// ------------------------------------------------------------------ k_steps_tile: ONE grid barrier per time step (D2Q9)
// The three phases of a step need two exchanges between SMs because psi(rho) of the new time level must be known at the
// eight neighbours before the force can be formed (and, next to walls, the virtual density of a boundary solid averages
// rho over ITS fluid neighbours, Eq. 17: a reach of two cells).  Here a CTA owns a TW x TH tile, one cell per thread, and
// recomputes rho and psi on a ring of H cells around it (H = 1 on fully periodic domains without solid cells, 2 otherwise)
// from the populations themselves -- the one-pass idea of K2F (lbm_fused_ws.cuh) on a 2-D tile:
//
//   A  every position of the (TW + 2H) x (TH + 2H) region: pull, rho (S1), psi (S3) into shared memory; the thread keeps
//      the populations of its own cell in registers
//   B  (masked / walled domains) solid positions of the inner ring: virtual density from the shared rho (S2, Eq. 17), psi
//   C  own cell: j, force from the shared psi (S4, S5), collide (S6), boundary rules and store (S7)
//   -- grid barrier, buffers swapped --
//
// so a step costs one trip through L2 and one grid barrier instead of two or three of each.  The ring is 27 % (H = 1,
// 16 x 16) to 41 % (H = 2, 32 x 16) more pulls, all L2 hits.  Same device functions and the same order of every sum as
// k_moments_v / k_virtual_density / k_step_v: bit-identical to the plain launches (tested).  The global rho / psi fields
// are not written (every entry point that reads them refreshes them first, as after the one-pass kernels).
// Positions beyond a non-periodic face do not exist: the neighbour offsets of an edge cell are clamped as in make_cell.
// TW x TH cells per CTA, CPT of them per thread
template <int TW, int TH, int CPT, bool BND>
struct SmallTile {
    static constexpr int H = BND ? 2 : 1;
    static constexpr int RW = TW + 2 * H, RH = TH + 2 * H;
    static constexpr int NCELL = TW * TH;
    static constexpr int NPOS = RW * RH;
    // one cell per thread: extra threads for the ring where they fit, so that every pull of phase A is in flight at once
    static constexpr int NT = CPT == 1 ? ((NPOS + 31) / 32 * 32 <= 1024 ? (NPOS + 31) / 32 * 32 : NCELL) : NCELL / CPT;
    static constexpr int NR = (NPOS + NT - 1) / NT;       // positions per thread in phase A (the first CPT are its own cells)
    static_assert(NCELL % CPT == 0 && NT % 32 == 0 && NT <= 1024, "whole warps");
    template <class CT> static constexpr size_t smem(int nc, int q) {
        return (size_t)NPOS * (sizeof(CT) * nc * (BND ? 2 : 1) + 4 + (BND ? 4 : 0) + 4 * q);
    }
};

template <class L, int NC, class CT, class ST, int COLL, bool BND, int TW, int TH, int CPT>
__global__ void __launch_bounds__((SmallTile<TW, TH, CPT, BND>::NT), 1)
k_steps_tile(const __grid_constant__ KParams<CT> p, int nsteps, unsigned* ctr) {
    static_assert(L::D == 2 && COLL != 2, "2-D lattices, with a collision");
    using T = SmallTile<TW, TH, CPT, BND>;
    constexpr int H = T::H, RW = T::RW, NPOS = T::NPOS, NT = T::NT, NR = T::NR, Q = L::Q;
    extern __shared__ __align__(16) unsigned char smem_t[];
    CT* psi_s = reinterpret_cast<CT*>(smem_t);                              // [NC][NPOS]
    CT* rho_s = psi_s + (BND ? NC * NPOS : 0);                              // [NC][NPOS] (walled domains)
    int* gid_s = reinterpret_cast<int*>(psi_s + (BND ? 2 : 1) * NC * NPOS); // global cell of a position, -1: none
    uint32_t* fl_s = reinterpret_cast<uint32_t*>(gid_s + NPOS);             // its flags (walled domains)
    uint32_t* src_s = fl_s + (BND ? NPOS : 0);                              // [Q][NPOS] element a pull reads, within a component

    const int tid = threadIdx.x;
    const int tiles_x = (p.nx + TW - 1) / TW;
    const int x0 = (int)(blockIdx.x % tiles_x) * TW, y0 = (int)(blockIdx.x / tiles_x) * TH;
    // position -> global cell (wrap on periodic axes; nothing beyond a non-periodic face), once
    int has_solid = 0;
    for (int pos = tid; pos < NPOS; pos += NT) {
        int gx = x0 + pos % RW - H, gy = y0 + pos / RW - H;
        bool ok = true;
        if (gx < 0) { if (p.periodic[0]) gx += p.nx; else ok = false; }
        else if (gx >= p.nx) { if (p.periodic[0]) gx -= p.nx; else ok = false; }
        if (gy < 0) { if (p.periodic[1]) gy += p.ny; else ok = false; }
        else if (gy >= p.ny) { if (p.periodic[1]) gy -= p.ny; else ok = false; }
        ok = ok && gx >= 0 && gx < p.nx && gy >= 0 && gy < p.ny;     // (domains narrower than the ring)
        const int g = ok ? gy * p.nx + gx : -1;
        gid_s[pos] = g;
        uint32_t fl = 0;
        if constexpr (BND) {
            fl = ok ? __ldg(p.flags + g) : SOLID_BIT;
            fl_s[pos] = fl;
            has_solid |= ok && (fl & SOLID_BIT) != 0;
        }
        // S7 read side as pull(): stored_i(x - e_i), or stored_ibar(x) on a flagged link -- the element index, once
        if (ok && !(fl & SOLID_BIT)) {
            const Cell c = make_cell<L>(p, g);
            static_for<0, Q>([&](auto I) {
                constexpr int i = I;
                constexpr int ib = opposite<L>(i);
                long long e = (long long)i * p.plane + g;
                if constexpr (i > 0) {
                    if (BND && ((fl >> i) & 1u)) e = (long long)ib * p.plane + g;
                    else e += nbr_offset<-L::E[i][0], -L::E[i][1], -L::E[i][2]>(c);
                }
                src_s[i * NPOS + pos] = (uint32_t)e;
            });
        }
    }
    // phase B is skipped by CTAs whose region holds no solid cell
    const int any_solid = __syncthreads_or(has_solid);     // (also the barrier between writing and reading gid_s / fl_s)
    const bool do_b = BND && any_solid && p.nbsolid > 0;
    // the e-th position of the region: the cells of the tile first (row by row), then the ring around it
    auto pos_of = [&](int e) {
        if (e < T::NCELL) return (e / TW + H) * RW + e % TW + H;
        int b = e - T::NCELL;
        if (b < H * RW) return b;                                                 // rows above
        b -= H * RW;
        if (b < TH * 2 * H) { const int r = b / (2 * H), c = b % (2 * H); return (H + r) * RW + (c < H ? c : TW + c); }
        b -= TH * 2 * H;
        return (H + TH) * RW + b;                                                 // rows below
    };
    // this thread's positions in phase A; bit r of `live`: a fluid cell of the domain sits there
    int posr[NR];
    unsigned live = 0, mine = 0;
    unsigned lofs[CPT];                 // own cells: bits 0..3 = the neighbour at x-1, x+1, y-1, y+1 is another position
#pragma unroll
    for (int r = 0; r < NR; ++r) {
        const int e = tid + r * NT;
        posr[r] = e < NPOS ? pos_of(e) : 0;
        bool ok = e < NPOS && gid_s[posr[r]] >= 0;
        if constexpr (BND) ok = ok && !(fl_s[posr[r]] & SOLID_BIT);
        if (ok) live |= 1u << r;
        // own cell of the tile AND inside the domain as such (a ragged tile's positions beyond the edge only serve as ring)
        if (r < CPT) {
            lofs[r] = 0;
            if (ok && e < T::NCELL && x0 + e % TW < p.nx && y0 + e / TW < p.ny) {
                mine |= 1u << r;
                const Cell c = make_cell<L>(p, gid_s[posr[r]]);
                lofs[r] = (c.sxm != 0 ? 1u : 0u) | (c.sxp != 0 ? 2u : 0u) | (c.sym != 0 ? 4u : 0u) | (c.syp != 0 ? 8u : 0u);
            }
        }
    }

    const ST* fa = static_cast<const ST*>(p.f_in);
    ST* fb = static_cast<ST*>(p.f_out);
    unsigned target = 0;
    for (int s = 0; s < nsteps; ++s) {
        // ---- A: pull at every position of the thread (all loads in flight together), then rho, psi into shared memory;
        //         the populations of the own cells stay in registers
        CT f[CPT][NC][Q];
        static_for<0, NR>([&](auto R) {
            constexpr int r = R;
            if ((live >> r) & 1u) {
                const int pos = posr[r];
#pragma unroll
                for (int k = 0; k < NC; ++k) {
                    CT tmp[Q];
                    const ST* base = fa + (long long)k * Q * p.plane;
                    static_for<0, Q>([&](auto I) { tmp[I] = CgLoad<CT, ST>::ld(base + src_s[I * NPOS + pos]) + p.wref[I]; });
                    const CT rr = density<L, CT>(tmp);
                    psi_s[k * NPOS + pos] = psi_of_rho(p, k, rr);
                    if constexpr (BND) rho_s[k * NPOS + pos] = rr;
                    if constexpr (r < CPT) {
#pragma unroll
                        for (int i = 0; i < Q; ++i) f[r][k][i] = tmp[i];
                    }
                }
            }
        });
        __syncthreads();
        // ---- B: virtual density at the solid positions of the tile and its inner ring (S2, Eq. 17; as k_virtual_density)
        if constexpr (BND) {
            if (do_b) {
                constexpr int IW = TW + 2, IH = TH + 2;
                for (int q = tid; q < IW * IH; q += NT) {
                    const int pos = (H - 1 + q / IW) * RW + (H - 1) + q % IW;
                    const int g = gid_s[pos];
                    if (g < 0 || !(fl_s[pos] & SOLID_BIT)) continue;
                    const Cell c = make_cell<L>(p, g);
                    const int dxm = c.sxm != 0 ? -1 : 0, dxp = c.sxp != 0 ? 1 : 0, dym = c.sym != 0 ? -RW : 0, dyp = c.syp != 0 ? RW : 0;
                    CT num[NC], den = CT(0);
#pragma unroll
                    for (int k = 0; k < NC; ++k) num[k] = CT(0);
                    static_for<1, Q>([&](auto I) {
                        constexpr int i = I;
                        constexpr CT w = CT(L::WN[i]) / CT(L::WD);
                        constexpr int ex = L::E[i][0], ey = L::E[i][1];
                        const int nb = pos + (ex > 0 ? dxp : (ex < 0 ? dxm : 0)) + (ey > 0 ? dyp : (ey < 0 ? dym : 0));
                        if (!(fl_s[nb] & SOLID_BIT)) {
                            den += w;
#pragma unroll
                            for (int k = 0; k < NC; ++k) num[k] += w * rho_s[k * NPOS + nb];
                        }
                    });
                    if (den > CT(0)) {
#pragma unroll
                        for (int k = 0; k < NC; ++k) {
                            CT rs = p.wet_phi[k] * (num[k] / den) - p.wet_drho[k];
                            rs = rs < p.wet_lo[k] ? p.wet_lo[k] : rs;
                            rs = rs > p.wet_hi[k] ? p.wet_hi[k] : rs;
                            psi_s[k * NPOS + pos] = psi_of_rho(p, k, rs);
                        }
                    }
                }
                __syncthreads();
            }
        }
        // ---- C: own cells (as k_step_v)
#pragma unroll
        for (int r = 0; r < CPT; ++r) {
            if (!((mine >> r) & 1u)) continue;
            const int own = posr[r];
            uint32_t own_fl = 0;
            if constexpr (BND) own_fl = fl_s[own];
            // local neighbour offsets (clamped at non-periodic faces like Cell::sxm ..), packed before the step loop
            const int lxm = -(int)((lofs[r] >> 0) & 1u), lxp = (int)((lofs[r] >> 1) & 1u);
            const int lym = ((lofs[r] >> 2) & 1u) ? -RW : 0, lyp = ((lofs[r] >> 3) & 1u) ? RW : 0;
            const int own_id = gid_s[own];
            CT rho[NC], j[NC][3];
#pragma unroll
            for (int k = 0; k < NC; ++k) moments<L, CT>(f[r][k], rho[k], j[k]);
            CT u[3] = {CT(0), CT(0), CT(0)}, du[NC][3];
            CT S[NC][3], pc[NC];
#pragma unroll
            for (int kp = 0; kp < NC; ++kp) {
                const CT* ps = psi_s + kp * NPOS + own;
                auto rowfn = [&](auto DY, auto DZ, auto NX, CT (&t)[1], CT& left, CT& right) {
                    constexpr int dy = DY;
                    const CT* row = ps + (dy > 0 ? lyp : (dy < 0 ? lym : 0));
                    t[0] = row[0];
                    if constexpr (NX != 0) { left = row[lxm]; right = row[lxp]; }
                };
                CT S1[3][1], pc1[1];
                psi_sums_rows<L, CT, 1>(rowfn, S1, pc1);
                S[kp][0] = S1[0][0]; S[kp][1] = S1[1][0]; S[kp][2] = S1[2][0];
                pc[kp] = pc1[0];
            }
            force_and_velocity<NC, CT>(p, rho, j, S, pc, u, du);
#pragma unroll
            for (int k = 0; k < NC; ++k) {
                collide<L, COLL, CT>(p, k, rho[k], u, du[k], f[r][k]);
                if constexpr (BND) {
                    if (own_fl & FACEBC_BIT) apply_face_rules<L, CT>(p, make_cell<L>(p, own_id), k, u, f[r][k]);
                }
                ST* out = fb + (long long)k * Q * p.plane + own_id;
                static_for<0, Q>([&](auto I) { Conv<CT, ST>::st(out + (long long)I * p.plane, f[r][k][I] - p.wref[I]); });
            }
        }
        grid_barrier(ctr, target, gridDim.x);       // (its __syncthreads also fences the shared fields for the next step)
        const ST* t_ = fa; fa = fb; fb = const_cast<ST*>(t_);
    }
}

}  // namespace lbmk
