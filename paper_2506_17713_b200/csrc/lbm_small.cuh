// lbm_small.cuh -- the two-pass step of small, launch-bound domains as ONE persistent kernel for n time steps.
//
//   k_steps_coop   n x [ K1: rho, psi  |  grid barrier  |  K1b: virtual density  |  grid barrier  |  K2: stream, force,
//                        collide, boundaries  |  grid barrier ]          (S1..S7; citations as in lbm_hot.cuh)
//
// Configs 1 and 2 (0.3 MB and 9.4 MB of state) live in L2 and a step is two or three kernels of a few microseconds: what
// a step costs there is the launch and drain of each kernel, even when replayed from a CUDA graph with programmatic
// dependent launches (11.5 us per step on config 2, 5 us on config 1).  Here the CTAs stay resident (cooperative launch),
// keep their cells for all n steps, and meet at a grid barrier between the phases: one atomic per CTA on a monotonic
// counter, polled with acquire loads.  Everything a phase reads was written by other SMs in the phase before, so global
// data is loaded with ld.global.cg (L2 only; the read-only path of the other kernels could serve stale L1 lines).
// Used where every cell gets its own resident thread (config 1: 4.8 -> 4.3 us per step; on config 2, where a thread would
// take two cells in turn, the separate vectorised kernels stay faster: 11.3 against 14.2 us, so the graph path remains).
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

}  // namespace lbmk
