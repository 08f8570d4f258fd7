// Fluid-compact layout of the two-pass path for porous domains (DESIGN.md 6 "Compact mode").
//
// With most cells solid (config 4: 77 %), the dense [cell] planes spend most of every 32-byte sector on solid slots that
// nobody reads.  While lbm_step runs on such a domain the populations therefore live in the order of the fluid-cell list:
// slot n of a direction plane belongs to the n-th fluid cell (brick order, lbm_api.cu; the planes are cplane = nfluid rounded
// up to 64 elements apart, so the whole state is one contiguous block), and psi lives in "extended" order
// (slots [0, nfluid) = fluid cells, [nfluid, nfluid + nbsolid) = boundary solids in the order of their list).
// In this layout the planes hold the POST-STREAM populations f_i(x_n, t) ("push" streaming): K1 and K2 read nothing but
// their own slot of every plane -- coalesced, no index in front of the loads -- and K2 scatters f*_i to the slot of the
// cell at x + e_i, or, when that cell is not fluid (halfway bounce-back, faces), to its own slot of plane ibar.  One
// neighbour table nbr[(i-1) * nbr_stride + n] (i = 1 .. Q-1) holds, in its low 28 bits, the extended index of the cell at
// x + e_i (wrap, or the clamped cell of R10; when the link crosses a non-periodic face bit 31 is set and bits 28-30 name the
// face, lowest axis first); K2 alone reads it, for the psi gather psi_ext[nbr[i] & NBR_IDX], as the scatter address and
// for the velocity / pressure rules of face links (no cell coordinates, flags or fluid list in the hot loop).  Every slot of a plane is written exactly once per step
// (by the one cell that streams or bounces into it), so the scatter is race-free and leaves no stale value.
// The arithmetic is the dense kernels' (same device functions, same order), so the results are bit-identical to the
// dense layout; every other entry point works on the dense layout, whose planes hold post-collision values at the
// writing cell (lbm_core.cuh): k_pack_c pulls them into compact order, k_unpack_c scatters them back.
#pragma once
#include "lbm_fused_ws.cuh"   // mbarrier / bulk-copy primitives

namespace lbmk {

constexpr uint32_t NBR_FACE = 0x80000000u;   // the link crosses a non-periodic face ...
constexpr int NBR_FACE_SHIFT = 28;          // ... this one (3 bits)
constexpr uint32_t NBR_IDX = 0x0fffffffu;    // extended index of the neighbour

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
        int face = -1;   // lowest axis first, as crossed_face() and the oracle's pull_source
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            if (pc[a] < 0) {
                if (p.periodic[a]) pc[a] += dims[a];
                else { pc[a] = 0; if (face < 0) face = 2 * a; }
            } else if (pc[a] >= dims[a]) {
                if (p.periodic[a]) pc[a] -= dims[a];
                else { pc[a] = dims[a] - 1; if (face < 0) face = 2 * a + 1; }
            }
        }
        const uint32_t e = (uint32_t)__ldg(cmap + pc[0] + p.nx * (pc[1] + p.ny * pc[2]));
        nbr[(long long)(i - 1) * p.nbr_stride + n] = (e & NBR_IDX) | (face >= 0 ? NBR_FACE | ((uint32_t)face << NBR_FACE_SHIFT) : 0u);
    });
}

// per boundary solid: fluid-list index of each neighbour (0xffffffff: not fluid), from the dense -> extended index map
template <class L, class CT>
__global__ void __launch_bounds__(256) k_build_snbr(const __grid_constant__ KParams<CT> p, const int* __restrict__ cmap,
                                                   uint32_t* __restrict__ snbr) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= p.nbsolid) return;
    const int id = __ldg(p.bsolid + b);
    const Cell c = make_cell<L>(p, id);
    static_for<1, L::Q>([&](auto I) {
        constexpr int i = I;
        const uint32_t e = (uint32_t)__ldg(cmap + id + nbr_offset<L::E[i][0], L::E[i][1], L::E[i][2]>(c));
        snbr[(long long)(i - 1) * p.snbr_stride + b] = e < (uint32_t)p.nfluid ? e : 0xffffffffu;
    });
}

// K1b in compact order (S2, Eq. 17): rho of the fluid neighbours from the compact rho field K1 wrote (coalesced
// table rows, gathers that stay in L2) instead of 18 scattered reads of the dense field; same operations in the same
// order as k_virtual_density
template <class L, int NC, class CT>
__global__ void __launch_bounds__(128) k_virtual_density_c(const __grid_constant__ KParams<CT> p) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= p.nbsolid) return;
    CT num[NC], den = CT(0);
#pragma unroll
    for (int k = 0; k < NC; ++k) num[k] = CT(0);
    uint32_t e[L::Q];
    static_for<1, L::Q>([&](auto I) { e[I] = __ldg(p.snbr + (long long)(I - 1) * p.snbr_stride + b); });
    static_for<1, L::Q>([&](auto I) {
        constexpr int i = I;
        constexpr CT w = CT(L::WN[i]) / CT(L::WD);
        if (e[i] != 0xffffffffu) {
            den += w;
#pragma unroll
            for (int k = 0; k < NC; ++k) num[k] += w * __ldg(p.rho + (long long)k * p.N + e[i]);
        }
    });
#pragma unroll
    for (int k = 0; k < NC; ++k) {
        CT rs = p.wet_phi[k] * (num[k] / den) - p.wet_drho[k];
        rs = rs < p.wet_lo[k] ? p.wet_lo[k] : rs;
        rs = rs > p.wet_hi[k] ? p.wet_hi[k] : rs;
        p.psi[(long long)k * p.N + p.nfluid + b] = psi_of_rho(p, k, rs);
    }
}

static __global__ void __launch_bounds__(256) k_cmap_scatter(int n, const int* __restrict__ list, int base, int* __restrict__ cmap) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t < n) cmap[list[t]] = base + t;
}

// dense (post-collision at the writing cell) -> compact (post-stream): the pull of lbm_core.cuh on raw storage values
template <class L, int NC, class CT, class ST>
__global__ void __launch_bounds__(256) k_pack_c(const __grid_constant__ KParams<CT> p) {
    const int n = blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= p.nfluid) return;
    const int id = __ldg(p.flist + n);
    const uint32_t fl = __ldg(p.flags + id);
    const Cell c = make_cell<L>(p, id);
#pragma unroll
    for (int k = 0; k < NC; ++k) {
        const ST* in = static_cast<const ST*>(p.f_in) + (long long)k * L::Q * p.plane + id;
        ST* out = static_cast<ST*>(p.f_out) + (long long)k * L::Q * p.cplane + n;
        static_for<0, L::Q>([&](auto I) {
            constexpr int i = I;
            constexpr int ib = opposite<L>(i);
            if constexpr (i == 0) out[0] = in[0];
            else out[(long long)i * p.cplane] = ((fl >> i) & 1u) ? in[(long long)ib * p.plane]
                                                                   : in[(long long)i * p.plane + nbr_offset<-L::E[i][0], -L::E[i][1], -L::E[i][2]>(c)];
        });
    }
}

// compact (post-stream) -> dense (post-collision at the writing cell): the scatter of k_unstream; every fluid slot of the
// dense planes is written exactly once, the solid ones by k_fill_solid
template <class L, int NC, class CT, class ST>
__global__ void __launch_bounds__(256) k_unpack_c(const __grid_constant__ KParams<CT> p) {
    const int n = blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= p.nfluid) return;
    const int id = __ldg(p.flist + n);
    const uint32_t fl = __ldg(p.flags + id);
    const Cell c = make_cell<L>(p, id);
#pragma unroll
    for (int k = 0; k < NC; ++k) {
        const ST* in = static_cast<const ST*>(p.f_in) + (long long)k * L::Q * p.cplane + n;
        ST* out = static_cast<ST*>(p.f_out) + (long long)k * L::Q * p.plane + id;
        static_for<0, L::Q>([&](auto I) {
            constexpr int i = I;
            constexpr int ib = opposite<L>(i);
            const ST v = in[(long long)i * p.cplane];
            if constexpr (i == 0) out[0] = v;
            else if ((fl >> i) & 1u) out[(long long)ib * p.plane] = v;
            else out[(long long)i * p.plane + nbr_offset<-L::E[i][0], -L::E[i][1], -L::E[i][2]>(c)] = v;
        });
    }
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

// the Q populations that have arrived at fluid cell n: its own slot of every plane
template <class L, class CT, class ST, bool WREF>
__device__ __forceinline__ void load_compact(const KParams<CT>& p, unsigned n, int k, CT (&f)[L::Q]) {
    // 32-bit element offsets within a component (Q * cplane < 2^32 is a condition of the mode)
    const ST* base = static_cast<const ST*>(p.f_in) + (long long)k * L::Q * p.cplane;
    const uint32_t cp = (uint32_t)p.cplane;
    static_for<0, L::Q>([&](auto I) {
        f[I] = ld_one<CT, ST>(base + ((uint32_t)I * cp + n));
        if constexpr (WREF) f[I] += p.wref[I];
    });
}

// ------------------------------------------------------------------ K1 in compact order: a streaming read, no table
template <class L, int NC, class CT, class ST, bool WREF>
__global__ void __launch_bounds__(256, 4) k_moments_c(const __grid_constant__ KParams<CT> p) {
    const unsigned n = blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= (unsigned)p.nfluid) return;
    // rho for K1b: in compact order when K1b has its neighbour table (snbr), else scattered into the dense field
    const int id = !p.write_rho ? 0 : (p.snbr ? (int)n : __ldg(p.flist + n));
#pragma unroll
    for (int k = 0; k < NC; ++k) {
        CT f[L::Q];
        load_compact<L, CT, ST, WREF>(p, n, k, f);
        const CT r = density<L, CT>(f);
        p.psi[(long long)k * p.N + n] = psi_of_rho(p, k, r);
        if (p.write_rho) p.rho[(long long)k * p.N + id] = r;
    }
}

// ... with 16-bit storage: two consecutive fluid cells per thread, so that a warp's request is 128 bytes again (one cell per
// thread made 38 half-sector loads per cell and ran at 4.5 TB/s where the fp32 kernel runs at 6.7)
template <class L, int NC, class CT, class ST, bool WREF>
__global__ void __launch_bounds__(256, 4) k_moments_c2(const __grid_constant__ KParams<CT> p) {
    static_assert(sizeof(ST) == 2, "the pair kernel is for 16-bit storage");
    const unsigned n = (blockIdx.x * blockDim.x + threadIdx.x) * 2u;      // cplane is a multiple of 64: n + 1 stays inside the plane
    if (n >= (unsigned)p.nfluid) return;
    const bool two = n + 1 < (unsigned)p.nfluid;
    const uint32_t cp = (uint32_t)p.cplane;
#pragma unroll
    for (int k = 0; k < NC; ++k) {
        const ST* base = static_cast<const ST*>(p.f_in) + (long long)k * L::Q * p.cplane;
        CT f0[L::Q], f1[L::Q];
        static_for<0, L::Q>([&](auto I) {
            CT t[2];
            ld_vec<CT, ST, 2>(base + ((uint32_t)I * cp + n), t);
            f0[I] = t[0]; f1[I] = t[1];
            if constexpr (WREF) { f0[I] += p.wref[I]; f1[I] += p.wref[I]; }
        });
        const CT r0 = density<L, CT>(f0), r1 = density<L, CT>(f1);
        CT* ps = p.psi + (long long)k * p.N + n;
        ps[0] = psi_of_rho(p, k, r0);
        if (two) ps[1] = psi_of_rho(p, k, r1);
        if (p.write_rho) {
            if (p.snbr) {
                CT* rr = p.rho + (long long)k * p.N + n;
                rr[0] = r0;
                if (two) rr[1] = r1;
            } else {
                p.rho[(long long)k * p.N + __ldg(p.flist + n)] = r0;
                if (two) p.rho[(long long)k * p.N + __ldg(p.flist + n + 1)] = r1;
            }
        }
    }
}

// ------------------------------------------------------------------ K2 in compact order
// A CTA owns CB consecutive fluid cells.  In compact order its Q populations per component and its Q-1 table rows are
// NC*Q + Q-1 contiguous runs of CB elements: they are brought into shared memory by bulk asynchronous copies (TMA unit,
// one request per run, all in flight at once, no registers), where the direct loads needed three dependent round
// trips under the register cap (table + first component, second component, psi gathers) and 40 % of the instructions
// were address arithmetic (profiles/r02_*).  What hangs on the table -- the psi gathers and the scatter addresses -- is
// issued as soon as the copies have landed; several CTAs per SM hide that second round trip.
template <class L, int NC, class ST>
struct CompactTile {
    // cells per CTA = threads, CTAs per SM (measured on config 4, K2: fp32 store 256 x 3 1.18 ms, 128 x 7 1.27, 128 x 8 1.42;
    // fp16 store 128 x 7 0.89 ms, 256 x 3 1.04)
    static constexpr int CB = sizeof(ST) == 2 ? 128 : 256;
    static constexpr int CTAS = sizeof(ST) == 2 ? 7 : 3;
    static constexpr int CPW = (NC * L::Q + L::Q - 1 + CB / 32 - 1) / (CB / 32);   // copies issued per warp (its first lanes)
    static constexpr int NPOP = NC * L::Q;                          // population runs
    static constexpr int NTAB = L::Q - 1;                           // table rows
    static constexpr size_t POP_BYTES = (size_t)NPOP * CB * sizeof(ST);
    static constexpr size_t TAB_BYTES = (size_t)NTAB * CB * 4;
    static constexpr size_t SMEM = POP_BYTES + TAB_BYTES + 16;
};

// WREF: populations are stored shifted by w_i rho_ref (R16)
template <class L, int NC, class CT, class ST, int COLL, bool WREF>
__global__ void __launch_bounds__((CompactTile<L, NC, ST>::CB), (CompactTile<L, NC, ST>::CTAS)) k_step_c(const __grid_constant__ KParams<CT> p) {
    using T = CompactTile<L, NC, ST>;
    constexpr int Q = L::Q, CB = T::CB;
    extern __shared__ __align__(16) unsigned char smem_c[];
    ST* pops = reinterpret_cast<ST*>(smem_c);                                   // [NC * Q][CB]
    uint32_t* tab = reinterpret_cast<uint32_t*>(smem_c + T::POP_BYTES);         // [Q - 1][CB]
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem_c + T::POP_BYTES + T::TAB_BYTES);
    const unsigned n0 = blockIdx.x * CB;
    const unsigned t = threadIdx.x;
    const unsigned n = n0 + t;
    // the planes are padded to cplane (a multiple of 64 elements), so the last CTA may copy up to the padded end
    const unsigned cnt = min((unsigned)CB, (unsigned)p.cplane - n0);
    if (t == 0) {
        mbar_init(bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (t == 0) mbar_expect_tx(bar, cnt * (uint32_t)(T::NPOP * sizeof(ST) + T::NTAB * 4));
    __syncthreads();
    {   // every warp issues CPW of the NPOP + NTAB copies (the issue loop is serial within a warp)
        const int lane = t & 31, c = (int)(t >> 5) * T::CPW + lane;
        if (lane < T::CPW && c < T::NPOP) {
            bulk_g2s(pops + c * CB, static_cast<const ST*>(p.f_in) + ((long long)c * p.cplane + n0), cnt * (uint32_t)sizeof(ST), bar);
        } else if (lane < T::CPW && c < T::NPOP + T::NTAB) {
            const int i = c - T::NPOP;
            bulk_g2s(tab + i * CB, p.nbr + ((long long)i * p.nbr_stride + n0), cnt * 4u, bar);
        }
    }
    mbar_wait(bar, 0);
    if (n >= (unsigned)p.nfluid) return;

    uint32_t nb[Q];
    nb[0] = n;
    static_for<1, Q>([&](auto I) { nb[I] = tab[(I - 1) * CB + t]; });
    // psi gathers first: the second (and last) round trip to memory
    CT S[NC][3], pc[NC];
    if constexpr (COLL != 2) {
#pragma unroll
        for (int kp = 0; kp < NC; ++kp) {
            const CT* ps = p.psi + (long long)kp * p.N;
            auto rowfn = [&](auto DY, auto DZ, auto NX, CT (&tv)[1], CT& left, CT& right) {
                constexpr int dy = DY, dz = DZ;
                if constexpr (dy == 0 && dz == 0) tv[0] = __ldg(ps + n);
                else if constexpr (row_has<L>(dy, dz, 0)) {
                    constexpr int i0 = dir_of<L>(0, dy, dz);   // constexpr locals: the lattice tables are host data
                    tv[0] = __ldg(ps + (nb[i0] & NBR_IDX));
                }
                if constexpr (NX != 0) {
                    constexpr int im = dir_of<L>(-1, dy, dz), ip = dir_of<L>(1, dy, dz);
                    left = __ldg(ps + (nb[im] & NBR_IDX));
                    right = __ldg(ps + (nb[ip] & NBR_IDX));
                }
            };
            CT S1[3][1], pc1[1];
            psi_sums_rows<L, CT, 1>(rowfn, S1, pc1);
            S[kp][0] = S1[0][0]; S[kp][1] = S1[1][0]; S[kp][2] = S1[2][0];
            pc[kp] = pc1[0];
        }
    }
    auto load_pops = [&](int k, CT (&fk)[Q]) {
        static_for<0, Q>([&](auto I) {
            fk[I] = Cvt<CT, ST>::up(pops[(k * Q + I) * CB + t]);
            if constexpr (WREF) fk[I] += p.wref[I];
        });
    };
    CT rho[NC], j[NC][3];
    CT u[3] = {CT(0), CT(0), CT(0)}, du[NC][3];
    if constexpr (COLL != 2) {
#pragma unroll
        for (int k = 0; k < NC; ++k) {
            CT fk[Q];
            load_pops(k, fk);
            moments<L, CT>(fk, rho[k], j[k]);
        }
        force_and_velocity<NC, CT>(p, rho, j, S, pc, u, du);
    }
    uint32_t anyface = 0;
    static_for<1, Q>([&](auto I) { anyface |= nb[I]; });
    // scatter offsets within a component (S7, push): f*_i goes to the cell at x + e_i, or bounces into the own slot of plane ibar
    const uint32_t cp = (uint32_t)p.cplane;
#pragma unroll
    for (int k = 0; k < NC; ++k) {
        CT fk[Q];
        load_pops(k, fk);
        if constexpr (COLL != 2) collide<L, COLL, CT>(p, k, rho[k], u, du[k], fk);
        if (anyface & NBR_FACE) {   // a link of this cell crosses a non-periodic face: velocity / pressure rules (R10)
            apply_face_rules_fn<L, CT>(p, [&](auto O) { return (nb[O] & NBR_FACE) ? (int)((nb[O] >> NBR_FACE_SHIFT) & 7u) : -1; }, k, u, fk);
        }
        ST* out = static_cast<ST*>(p.f_out) + (long long)k * Q * p.cplane;
        static_for<0, Q>([&](auto I) {
            constexpr int i = I;
            if constexpr (i == 0) {
                Conv<CT, ST>::st(out + n, WREF ? fk[0] - p.wref[0] : fk[0]);
            } else {
                constexpr int ib = opposite<L>(i);
                const uint32_t d = nb[i];
                const uint32_t off = d < (uint32_t)p.nfluid ? (uint32_t)i * cp + d : (uint32_t)ib * cp + n;
                Conv<CT, ST>::st(out + off, WREF ? fk[i] - p.wref[i] : fk[i]);   // (w_i = w_ibar)
            }
        });
    }
}

}  // namespace lbmk
