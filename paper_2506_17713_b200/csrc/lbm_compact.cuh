// Fluid-compact layout of the two-pass path for porous domains (DESIGN.md 6 "Compact mode").
//
// With most cells solid (config 4: 77 %), the dense [cell] planes spend most of every 32-byte sector on solid slots that
// nobody reads.  While lbm_step runs on such a domain the populations therefore live in the order of the fluid-cell list:
// slot n of a direction plane belongs to the n-th fluid cell (ascending cell index; the planes are cplane = nfluid rounded
// up to 64 elements apart, so the whole state is one contiguous block), and psi lives in "extended" order
// (slots [0, nfluid) = fluid cells, [nfluid, nfluid + nbsolid) = boundary solids in the order of their list).  One
// neighbour table nbr[(i-1) * nbr_stride + n] (i = 1 .. Q-1) holds the extended index of the cell at x + e_i (wrap, or the
// clamped cell of R10 with bit 31 set when the link crosses a non-periodic face).  It serves both stencils:
//   pull of direction i   : source x - e_i = x + e_ibar -> nbr[ibar]; a fluid index (< nfluid, bit 31 clear) is read,
//                           anything else is a flagged link (halfway bounce-back: own stored_ibar)
//   psi of neighbour x+e_i: psi_ext[nbr[i] & 0x7fffffff]
// The arithmetic is the dense kernels' (same device functions, same order), so the results are bit-identical to the
// dense layout; every other entry point works on the dense layout (k_pack / k_unpack convert at the boundary).
#pragma once
#include "lbm_hot.cuh"

namespace lbmk {

constexpr uint32_t NBR_FACE = 0x80000000u;

// neighbour table from the dense -> extended index map (cmap: -1 for solids that touch no fluid cell)
template <class L, class CT>
__global__ void __launch_bounds__(256) k_build_nbr(const __grid_constant__ KParams<CT> p, const int* __restrict__ cmap,
                                                  uint32_t* __restrict__ nbr) {
    const int n = blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= p.nfluid) return;
    const int id = __ldg(p.flist + n);
    const int x = id % p.nx, t = id / p.nx, y = t % p.ny, z = t / p.ny;
    const int dims[3] = {p.nx, p.ny, p.nz};
    static_for<1, L::Q>([&](auto I) {
        constexpr int i = I;
        int pc[3] = {x + L::E[i][0], y + L::E[i][1], z + L::E[i][2]};
        bool crossed = false;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            if (pc[a] < 0) {
                if (p.periodic[a]) pc[a] += dims[a];
                else { pc[a] = 0; crossed = true; }
            } else if (pc[a] >= dims[a]) {
                if (p.periodic[a]) pc[a] -= dims[a];
                else { pc[a] = dims[a] - 1; crossed = true; }
            }
        }
        const uint32_t e = (uint32_t)__ldg(cmap + pc[0] + p.nx * (pc[1] + p.ny * pc[2]));
        nbr[(long long)(i - 1) * p.nbr_stride + n] = (e & ~NBR_FACE) | (crossed ? NBR_FACE : 0u);
    });
}

static __global__ void __launch_bounds__(256) k_cmap_scatter(int n, const int* __restrict__ list, int base, int* __restrict__ cmap) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t < n) cmap[list[t]] = base + t;
}

// dense -> compact / compact -> dense copies of every population plane (T = raw storage element)
template <class T>
__global__ void __launch_bounds__(256) k_pack(const T* __restrict__ src, T* __restrict__ dst, const int* __restrict__ flist,
                                             int nfluid, long long plane, long long cplane, int nplanes, int to_dense) {
    const int n = blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= nfluid) return;
    const int id = __ldg(flist + n);
    const long long from = to_dense ? n : id, to = to_dense ? id : n;
    const long long sp = to_dense ? cplane : plane, dp = to_dense ? plane : cplane;
    for (int pl = 0; pl < nplanes; ++pl) dst[pl * dp + to] = src[pl * sp + from];
}

// solid cells of the dense layout hold f_eq(1, 0) (include/lbm.h, lbm_init_fields)
template <class L, int NC, class CT, class ST>
__global__ void __launch_bounds__(256) k_fill_solid(const __grid_constant__ KParams<CT> p) {
    const int id = blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= p.N || !(__ldg(p.flags + id) & SOLID_BIT)) return;
    const CT u[3] = {CT(0), CT(0), CT(0)};
#pragma unroll
    for (int k = 0; k < NC; ++k) {
        ST* out = static_cast<ST*>(p.f_out) + (long long)k * L::Q * p.plane + id;
        static_for<0, L::Q>([&](auto I) {
            constexpr int i = I;
            Conv<CT, ST>::st(out + (long long)i * p.plane, feq<L, i, CT>(CT(1), u, CT(0)) - p.wref[i]);
        });
    }
}

// the thread's row of the neighbour table
template <class L, class CT>
__device__ __forceinline__ void load_nbr(const KParams<CT>& p, unsigned n, uint32_t (&nb)[L::Q]) {
    nb[0] = n;
    static_for<1, L::Q>([&](auto I) { nb[I] = __ldg(p.nbr + (long long)(I - 1) * p.nbr_stride + n); });
}

// S7 read side in compact order: f[i] = stored_i(x - e_i), or stored_ibar(x) on a flagged link
template <class L, class CT, class ST>
__device__ __forceinline__ void pull_compact(const KParams<CT>& p, unsigned n, const uint32_t (&nb)[L::Q], int k, CT (&f)[L::Q]) {
    // 32-bit element offsets within a component (Q * cplane < 2^32 is a condition of the mode)
    const ST* base = static_cast<const ST*>(p.f_in) + (long long)k * L::Q * p.cplane;
    const uint32_t cp = (uint32_t)p.cplane;
    static_for<0, L::Q>([&](auto I) {
        constexpr int i = I;
        if constexpr (i == 0) {
            f[0] = ld_one<CT, ST>(base + n) + p.wref[0];
        } else {
            constexpr int ib = opposite<L>(i);
            const uint32_t s = nb[ib];
            const bool ok = s < (uint32_t)p.nfluid;
            const uint32_t off = ok ? (uint32_t)i * cp + s : (uint32_t)ib * cp + n;
            f[i] = ld_one<CT, ST>(base + off) + p.wref[i];
        }
    });
}

// ------------------------------------------------------------------ K1 in compact order
template <class L, int NC, class CT, class ST>
__global__ void __launch_bounds__(256, 4) k_moments_c(const __grid_constant__ KParams<CT> p) {
    const unsigned n = blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= (unsigned)p.nfluid) return;
    uint32_t nb[L::Q];
    load_nbr<L, CT>(p, n, nb);
    const int id = p.write_rho ? __ldg(p.flist + n) : 0;
#pragma unroll
    for (int k = 0; k < NC; ++k) {
        CT f[L::Q];
        pull_compact<L, CT, ST>(p, n, nb, k, f);
        const CT r = density<L, CT>(f);
        p.psi[(long long)k * p.N + n] = psi_of_rho(p, k, r);
        if (p.write_rho) p.rho[(long long)k * p.N + id] = r;   // dense: K1b averages it around the boundary solids
    }
}

// ------------------------------------------------------------------ K2 in compact order
// One cell per thread and gathers everywhere: the kernel lives on warps in flight.  With two components the 2 x Q
// pulled populations are parked in shared memory ([component][direction][thread], conflict-free, private to the
// thread: no barrier) between the moment sums and the collision, which keeps the kernel at 64 .. 100 registers
// (five to eight CTAs per SM instead of four at 128 registers).
#ifndef LBM_COMPACT_PARK
#define LBM_COMPACT_PARK 1
#endif
// CTAs per SM (measured on config 4, 400^3: fp32 store 1.46 ms at 5 against 1.52 at 8; fp16 store 1.29 at 8, 1.41 at 5)
#ifndef LBM_COMPACT_CTAS
#define LBM_COMPACT_CTAS (sizeof(ST) == 2 ? 8 : 5)
#endif
template <class L, int NC, class CT, class ST, int COLL>
__global__ void __launch_bounds__(128, ((NC == 2 && LBM_COMPACT_PARK) || sizeof(ST) == 2 ? LBM_COMPACT_CTAS : 1))
k_step_c(const __grid_constant__ KParams<CT> p) {
    constexpr bool PARK = NC == 2 && LBM_COMPACT_PARK;
    __shared__ CT park[PARK ? NC * L::Q * 128 : 1];
    const unsigned n = blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= (unsigned)p.nfluid) return;
    uint32_t nb[L::Q];
    load_nbr<L, CT>(p, n, nb);

    CT f[PARK ? 1 : NC][L::Q], rho[NC], j[NC][3];
#pragma unroll
    for (int k = 0; k < NC; ++k) {
        CT(&fk)[L::Q] = f[PARK ? 0 : k];
        pull_compact<L, CT, ST>(p, n, nb, k, fk);
        if constexpr (COLL != 2) moments<L, CT>(fk, rho[k], j[k]);
        if constexpr (PARK) static_for<0, L::Q>([&](auto I) { park[(k * L::Q + I) * 128 + threadIdx.x] = fk[I]; });
    }
    CT u[3] = {CT(0), CT(0), CT(0)}, du[NC][3];
    if constexpr (COLL != 2) {
        CT S[NC][3], pc[NC];
#pragma unroll
        for (int kp = 0; kp < NC; ++kp) {
            const CT* ps = p.psi + (long long)kp * p.N;
            auto rowfn = [&](auto DY, auto DZ, auto NX, CT (&t)[1], CT& left, CT& right) {
                constexpr int dy = DY, dz = DZ;
                if constexpr (dy == 0 && dz == 0) t[0] = __ldg(ps + n);
                else if constexpr (row_has<L>(dy, dz, 0)) {
                    constexpr int i0 = dir_of<L>(0, dy, dz);   // constexpr locals: the lattice tables are host data
                    t[0] = __ldg(ps + (nb[i0] & ~NBR_FACE));
                }
                if constexpr (NX != 0) {
                    constexpr int im = dir_of<L>(-1, dy, dz), ip = dir_of<L>(1, dy, dz);
                    left = __ldg(ps + (nb[im] & ~NBR_FACE));
                    right = __ldg(ps + (nb[ip] & ~NBR_FACE));
                }
            };
            CT S1[3][1], pc1[1];
            psi_sums_rows<L, CT, 1>(rowfn, S1, pc1);
            S[kp][0] = S1[0][0]; S[kp][1] = S1[1][0]; S[kp][2] = S1[2][0];
            pc[kp] = pc1[0];
        }
        force_and_velocity<NC, CT>(p, rho, j, S, pc, u, du);
    }
    uint32_t anyface = 0;
    static_for<1, L::Q>([&](auto I) { anyface |= nb[I]; });
#pragma unroll
    for (int k = 0; k < NC; ++k) {
        CT(&fk)[L::Q] = f[PARK ? 0 : k];
        if constexpr (PARK) static_for<0, L::Q>([&](auto I) { fk[I] = park[(k * L::Q + I) * 128 + threadIdx.x]; });
        if constexpr (COLL != 2) collide<L, COLL, CT>(p, k, rho[k], u, du[k], fk);
        if (anyface & NBR_FACE) {   // a link of this cell crosses a non-periodic face: velocity / pressure rules (R10)
            const int id = __ldg(p.flist + n);
            if (__ldg(p.flags + id) & FACEBC_BIT) {
                Cell cc;
                cc.x = id % p.nx; cc.y = (id / p.nx) % p.ny; cc.z = id / (p.nx * p.ny);
                apply_face_rules<L, CT>(p, cc, k, u, fk);
            }
        }
        ST* out = static_cast<ST*>(p.f_out) + (long long)k * L::Q * p.cplane;
        const uint32_t cp = (uint32_t)p.cplane;
        static_for<0, L::Q>([&](auto I) { Conv<CT, ST>::st(out + ((uint32_t)I * cp + n), fk[I] - p.wref[I]); });
    }
}

}  // namespace lbmk
