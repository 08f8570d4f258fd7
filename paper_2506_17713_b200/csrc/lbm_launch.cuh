// lbm_launch.cuh -- host-side dispatch from run-time options to the kernel templates of lbm_core.cuh.
// One translation unit per (lattice, compute dtype, storage dtype) instantiates launch<L,CT,ST>.
#pragma once
#include <cstdio>
#include <cstdlib>
#include "lbm_fused_ws.cuh"
#include "lbm_fused_eq.cuh"
#include <algorithm>
#include "lbm_fused_eq2.cuh"
#include "lbm_compact.cuh"
#include "lbm_small.cuh"

namespace lbmk {

enum Op { OP_MOMENTS = 0, OP_VIRTUAL = 1, OP_STEP = 2, OP_INIT = 3, OP_EXPORT_MACRO = 4, OP_EXPORT_POP = 5, OP_IMPORT_POP = 6, OP_UNSTREAM = 7, OP_FUSED = 8,
          OP_BUILD_NBR = 9 /* a0 = dense -> extended index map, a2 = table */, OP_FILL_SOLID = 10,
          OP_PACK_C = 11 /* dense -> compact layout */, OP_UNPACK_C = 12 /* compact -> dense */,
          OP_BUILD_SNBR = 13 /* a0 = dense -> extended index map, a2 = table of the boundary solids */,
          OP_COOP = 14 /* i0 = time steps, a2 = barrier counter (zeroed): the persistent kernel of small domains */,
          OP_TILE = 15 /* same arguments: the tiled persistent kernel of small 2-D domains (one barrier per step) */ };

struct LaunchArgs {
    int op;
    int nc;    // components
    int coll;  // 0 BGK, 1 MRT, 2 none (pure streaming)
    int vec;   // cells per thread along x in the hot kernels: 1 or vec_width<CT, ST, NC>() (needs nx % vec == 0)
    int list;  // 1: hot kernels iterate over the fluid-cell list (one cell per thread) instead of the whole grid;
               // 2: compact mode, populations in fluid-list order (lbm_compact.cuh)
    int zc;    // a component has a Zhang-Chen weight: K2 runs its one-cell-per-thread Zhang-Chen variant
    int bnd;   // any solid cell or non-periodic axis
    const void* params;  // KParams<CT>
    const void* a0;      // op-specific (FieldIO<CT>* for init / import / export_pop; u_out for export_macro)
    const void* a1;
    void* a2;
    int i0;              // op-specific integer (OP_FUSED: planes marched per CTA)
    int i1;              // OP_FUSED, k_fused_eq_split: tile rows per launch (0: the whole domain in one launch)
    int i2;              // OP_FUSED, k_fused_ws: rows per tile (0: the default of fused_shape)
    int eq;              // OP_FUSED: one component, BGK, tau = 1 (f* is an equilibrium): the row-pipeline kernel k_fused_eq applies
                         //           (2: with half-width tiles and two CTAs per SM; 3 / 4: k_fused_eq_split, late / early take)
    int* used_kernel;    // OP_FUSED, out: the lbm_path value of the kernel that ran
    int wref;            // OP_FUSED: rho_ref != 0 (populations stored shifted by w_i rho_ref)
    int pdl;             // OP_MOMENTS / OP_VIRTUAL / OP_STEP (dense mapping): programmatic dependent launch (pdl_begin)
    cudaStream_t stream;
};

// Tile of the one-pass kernels K2F (D3Q19) per (dtypes, components): VEC cells per lane (tile width 32 x VEC), TY rows.
// VEC = 0: no one-pass kernel built for this combination (the two-pass path is used).
struct FusedShape { int vec, ty; };
template <class L, class CT, class ST, int NC>
constexpr FusedShape fused_shape() {
    if (L::D != 3) return FusedShape{0, 0};
    if (sizeof(CT) == 4) return NC == 1 ? FusedShape{4, 8} : FusedShape{2, 8};
    return NC == 1 ? FusedShape{2, 8} : FusedShape{0, 0};
}

template <class L, class CT, class ST>
cudaError_t launch(const LaunchArgs& a);

// Widest per-thread vector of the hot kernels: 16-byte population accesses, capped so that the populations a
// thread holds (NC * Q * VEC values) stay within ~80 32-bit registers.
template <class CT, class ST, int NC>
constexpr int vec_width() {
    int v = 16 / (int)sizeof(ST);
    const int cap = 4 / (NC * ((int)sizeof(CT) / 4));   // fp32: 4 (NC=1), 2 (NC=2); fp64: 2, 1
    if (v > cap) v = cap;
    return v < 1 ? 1 : v;
}

#ifdef LBM_INSTANTIATE
template <class L, class CT, class ST>
cudaError_t launch(const LaunchArgs& a) {
    const KParams<CT>& p = *static_cast<const KParams<CT>*>(a.params);
    auto grid = [&](int n, int block) { return dim3((unsigned)((n + block - 1) / block)); };
    auto with_nc = [&](auto fn) {
        if (a.nc == 1) fn(IC<1>{});
        else fn(IC<2>{});
    };
    auto with_bnd = [&](auto fn) {
        if (a.bnd) fn(IC<1>{});
        else fn(IC<0>{});
    };
    // hot kernels of the dense mapping: plain launch, or with the programmatic-serialisation attribute (pdl_begin)
    auto launch_hot = [&](auto kernel, dim3 g, unsigned block) {
        if (!a.pdl) {
            kernel<<<g, block, 0, a.stream>>>(p);
            return;
        }
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = g;
        cfg.blockDim = dim3(block);
        cfg.stream = a.stream;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = at;
        cfg.numAttrs = 1;
        cudaLaunchKernelEx(&cfg, kernel, p);
    };
    switch (a.op) {
        case OP_MOMENTS:
            with_nc([&](auto NC) {
                with_bnd([&](auto B) {
                    constexpr int VW = vec_width<CT, ST, NC>();
                    if constexpr (B != 0) {
                        if (a.list == 2) {
                            if constexpr (sizeof(ST) == 2) {      // 16-bit storage: two cells per thread (32-bit loads)
                                if (a.wref) k_moments_c2<L, NC, CT, ST, true><<<grid((p.nfluid + 1) / 2, 256), 256, 0, a.stream>>>(p);
                                else k_moments_c2<L, NC, CT, ST, false><<<grid((p.nfluid + 1) / 2, 256), 256, 0, a.stream>>>(p);
                                return;
                            }
                            if (a.wref) k_moments_c<L, NC, CT, ST, true><<<grid(p.nfluid, 256), 256, 0, a.stream>>>(p);
                            else k_moments_c<L, NC, CT, ST, false><<<grid(p.nfluid, 256), 256, 0, a.stream>>>(p);
                            return;
                        }
                        if (a.list) {
                            k_moments_v<L, NC, CT, ST, true, 1, true><<<grid(p.nfluid, 256), 256, 0, a.stream>>>(p);
                            return;
                        }
                    }
                    if (a.vec == VW && VW > 1)
                        launch_hot(k_moments_v<L, NC, CT, ST, (B != 0), VW>, grid(p.N / VW, 256), 256);
                    else
                        launch_hot(k_moments_v<L, NC, CT, ST, (B != 0), 1>, grid(p.N, 256), 256);
                });
            });
            break;
        case OP_VIRTUAL:
            if (p.nbsolid > 0)
                with_nc([&](auto NC) {
                    if (p.compact && p.snbr) k_virtual_density_c<L, NC, CT><<<grid(p.nbsolid, 128), 128, 0, a.stream>>>(p);
                    else launch_hot(k_virtual_density<L, NC, CT>, grid(p.nbsolid, 128), 128);
                });
            break;
        case OP_STEP:
            with_nc([&](auto NC) {
                with_bnd([&](auto B) {
                    auto with_coll = [&](auto fn) {
                        if (a.coll == 0) fn(IC<0>{});
                        else if (a.coll == 1) fn(IC<1>{});
                        else fn(IC<2>{});
                    };
                    with_coll([&](auto C_) {
                        constexpr int VW = vec_width<CT, ST, NC>();
                        if constexpr (C_ != 2) {
                            if (a.zc) {
                                k_step_v<L, NC, CT, ST, C_, (B != 0), 1, false, true><<<grid(p.N, 128), 128, 0, a.stream>>>(p);
                                return;
                            }
                        }
                        if constexpr (B != 0) {
                            if (a.list == 2) {
                                using T = CompactTile<L, NC, ST>;
                                auto go_c = [&](auto kern) {
                                    if (T::SMEM > 48 * 1024) cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)T::SMEM);
                                    kern<<<grid(p.nfluid, T::CB), T::CB, T::SMEM, a.stream>>>(p);
                                };
                                if (a.wref) go_c(k_step_c<L, NC, CT, ST, C_, true>);
                                else go_c(k_step_c<L, NC, CT, ST, C_, false>);
                                return;
                            }
                            if (a.list) {
                                k_step_v<L, NC, CT, ST, C_, true, 1, true><<<grid(p.nfluid, 128), 128, 0, a.stream>>>(p);
                                return;
                            }
                        }
                        if (a.vec == VW && VW > 1)
                            launch_hot(k_step_v<L, NC, CT, ST, C_, (B != 0), VW>, grid(p.N / VW, 128), 128);
                        else
                            launch_hot(k_step_v<L, NC, CT, ST, C_, (B != 0), 1>, grid(p.N, 128), 128);
                    });
                });
            });
            break;
        case OP_BUILD_NBR:
            k_build_nbr<L, CT><<<grid(p.nfluid, 256), 256, 0, a.stream>>>(p, static_cast<const int*>(a.a0), static_cast<uint32_t*>(a.a2));
            break;
        case OP_COOP: {
            cudaError_t err = cudaErrorInvalidValue;
            with_nc([&](auto NC) {
                with_bnd([&](auto B) {
                    auto with_coll = [&](auto fn) {
                        if (a.coll == 0) fn(IC<0>{});
                        else if (a.coll == 1) fn(IC<1>{});
                        else fn(IC<2>{});
                    };
                    with_coll([&](auto C_) {
                        auto kern = k_steps_coop<L, NC, CT, ST, C_, (B != 0)>;
                        int dev = 0, nsm = 0, per_sm = 0, coop = 0;
                        cudaGetDevice(&dev);
                        cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
                        cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
                        if (!coop || cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, 256, 0) != cudaSuccess || per_sm < 1) {
                            err = cudaErrorNotSupported;
                            return;
                        }
                        // one cell per resident thread at most: with two cells in sequence per thread the phases take longer than
                        // the separate, vectorised kernels (measured on config 2, 131 072 cells: 14.2 against 11.3 us per step)
                        const int want = (p.N + 255) / 256;
                        if (want > nsm * per_sm) { err = cudaErrorNotSupported; return; }
                        const int g = want;
                        int nsteps = a.i0;
                        unsigned* ctr = static_cast<unsigned*>(a.a2);
                        void* args[] = {const_cast<void*>(static_cast<const void*>(&p)), &nsteps, &ctr};
                        err = cudaLaunchCooperativeKernel(reinterpret_cast<const void*>(kern), dim3((unsigned)g), dim3(256), args, 0, a.stream);
                    });
                });
            });
            if (err != cudaSuccess) { cudaGetLastError(); return err; }
            break;
        }
        case OP_TILE: {
            // k_steps_tile (lbm_small.cuh): one CTA per TW x TH tile, all resident, one grid barrier per step
            cudaError_t err = cudaErrorNotSupported;
            if constexpr (L::D == 2) {
                with_nc([&](auto NC) {
                    with_bnd([&](auto B) {
                        auto with_coll = [&](auto fn) {
                            if (a.coll == 0) fn(IC<0>{});
                            else if (a.coll == 1) fn(IC<1>{});
                        };
                        with_coll([&](auto C_) {
                            int dev = 0, nsm = 0, coop = 0;
                            cudaGetDevice(&dev);
                            cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
                            cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
                            if (!coop) return;
                            auto go = [&](auto TW_, auto TH_, auto CPT_) {
                                constexpr int TW = TW_, TH = TH_, CPT = CPT_;
                                using T = SmallTile<TW, TH, CPT, (B != 0)>;
                                auto kern = k_steps_tile<L, NC, CT, ST, C_, (B != 0), TW, TH, CPT>;
                                const size_t smem = T::template smem<CT>(NC, L::Q);
                                const int g = ((p.nx + TW - 1) / TW) * ((p.ny + TH - 1) / TH);
                                if (g > nsm) return false;          // one CTA per SM, all resident
                                int per_sm = 0;
                                if (smem > 48 * 1024 && cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return false;
                                if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, T::NT, smem) != cudaSuccess || per_sm < 1) return false;
                                int nsteps = a.i0;
                                unsigned* ctr = static_cast<unsigned*>(a.a2);
                                void* args[] = {const_cast<void*>(static_cast<const void*>(&p)), &nsteps, &ctr};
                                err = cudaLaunchCooperativeKernel(reinterpret_cast<const void*>(kern), dim3((unsigned)g), dim3(T::NT), args, smem, a.stream);
                                return true;
                            };
                            // the smallest tile that gives every SM at most one CTA, one cell per thread
                            if (go(IC<8>{}, IC<8>{}, IC<1>{})) return;
                            if (go(IC<16>{}, IC<16>{}, IC<1>{})) return;
                            if (go(IC<32>{}, IC<16>{}, IC<1>{})) return;
                            go(IC<64>{}, IC<16>{}, IC<1>{});
                        });
                    });
                });
            }
            if (err != cudaSuccess) { cudaGetLastError(); return err; }
            break;
        }
        case OP_BUILD_SNBR:
            k_build_snbr<L, CT><<<grid(p.nbsolid, 256), 256, 0, a.stream>>>(p, static_cast<const int*>(a.a0), static_cast<uint32_t*>(a.a2));
            break;
        case OP_FILL_SOLID:
            with_nc([&](auto NC) { k_fill_solid<L, NC, CT, ST><<<grid(p.N, 256), 256, 0, a.stream>>>(p); });
            break;
        case OP_PACK_C:
            with_nc([&](auto NC) { k_pack_c<L, NC, CT, ST><<<grid(p.nfluid, 256), 256, 0, a.stream>>>(p); });
            break;
        case OP_UNPACK_C:
            with_nc([&](auto NC) { k_unpack_c<L, NC, CT, ST><<<grid(p.nfluid, 256), 256, 0, a.stream>>>(p); });
            break;
        case OP_UNSTREAM:
            with_nc([&](auto NC) {
                with_bnd([&](auto B) {
                    k_unstream<L, NC, ST, CT, (B != 0)><<<grid(p.N, 256), 256, 0, a.stream>>>(p, a.i0);
                });
            });
            break;
        case OP_INIT: {
            const FieldIO<CT>& io = *static_cast<const FieldIO<CT>*>(a.a0);
            with_nc([&](auto NC) {
                k_init<L, NC, CT, ST><<<grid(io.cnt, 256), 256, 0, a.stream>>>(p, io, a.a2, a.i0);
            });
            break;
        }
        case OP_EXPORT_MACRO:
            with_nc([&](auto NC) {
                with_bnd([&](auto B) {
                    k_export_macro<L, NC, CT, ST, (B != 0)><<<grid(p.N, 128), 128, 0, a.stream>>>(
                        p, static_cast<CT*>(const_cast<void*>(a.a0)), static_cast<CT*>(const_cast<void*>(a.a1)));
                });
            });
            break;
        case OP_EXPORT_POP: {
            const FieldIO<CT>& io = *static_cast<const FieldIO<CT>*>(a.a0);
            with_bnd([&](auto B) {
                k_export_pop<L, CT, ST, (B != 0)><<<grid(io.cnt, 256), 256, 0, a.stream>>>(p, a.i0, io);
            });
            break;
        }
        case OP_IMPORT_POP: {
            const FieldIO<CT>& io = *static_cast<const FieldIO<CT>*>(a.a0);
            k_import_pop<L, CT, ST><<<grid(io.cnt, 256), 256, 0, a.stream>>>(p, a.i0, io, a.a2);
            break;
        }
        case OP_FUSED: {
            bool done = false;
            int dev = 0;
            cudaGetDevice(&dev);
            // dynamic shared memory opt-in and the register pool the kernels re-split with setmaxnreg (a smaller pool would make
            // setmaxnreg.inc wait forever): checked once per device and kernel
            auto usable = [&](auto kern, int (&ready)[16], size_t smem, long long regs_needed, int threads) {
                int& rd = ready[dev & 15];   // 0 unknown, 1 usable, -1 not usable
                if (rd == 0) {
                    cudaFuncAttributes fa;
                    const cudaError_t e1 = cudaFuncGetAttributes(&fa, kern);
                    const bool regs_ok = e1 == cudaSuccess && (long long)fa.numRegs * threads >= regs_needed;
                    const cudaError_t e2 = regs_ok ? cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)
                                                   : cudaErrorUnknown;
                    rd = (regs_ok && e2 == cudaSuccess) ? 1 : -1;
                    cudaGetLastError();
                }
                return rd > 0;
            };
            with_nc([&](auto NC) {
                auto with_coll = [&](auto fn) {
                    if (a.coll == 0) fn(IC<0>{});
                    else if (a.coll == 1) fn(IC<1>{});
                };
                with_coll([&](auto C_) {
                    constexpr FusedShape fs = fused_shape<L, CT, ST, NC>();
                    if constexpr (fs.vec > 0) {
                        // k_fused_ws: warp-specialised producer / consumer pipeline, two stages of fs.ty rows
                        // (TYW rows per tile: fs.ty, or one fewer where that gives every SM a CTA -- plan_fused, a.i2)
                        auto go_ws_ty = [&](auto WREF, auto TYW_) {
                            constexpr int TYW = TYW_;
                            using T = WsTile<L, NC, CT, ST, fs.vec, TYW, 2>;
                            auto kern = k_fused_ws<L, NC, CT, ST, C_, fs.vec, TYW, 2, (WREF != 0)>;
                            static int ready[16] = {0};
                            if (!usable(kern, ready, T::SMEM, (long long)T::REG_PROD * T::NPW * 32 + (long long)T::REG_CONS * T::NCW * 32, T::THREADS)) return;
                            dim3 g((unsigned)((p.nx + T::TX - 1) / T::TX), (unsigned)((p.ny + TYW - 1) / TYW),
                                   (unsigned)((p.nz + a.i0 - 1) / a.i0));
                            kern<<<g, T::THREADS, T::SMEM, a.stream>>>(p, a.i0);
                            if (a.used_kernel) *a.used_kernel = 3;  // LBM_PATH_ONE_PASS_WS
                            done = true;
                        };
                        auto go_ws = [&](auto WREF) {
                            if constexpr (NC == 1) {
                                if (a.i2 == fs.ty - 1) { go_ws_ty(WREF, IC<fs.ty - 1>{}); return; }
                            }
                            go_ws_ty(WREF, IC<fs.ty>{});
                        };
                        // k_fused_eq: row pipelines (lbm_fused_eq.cuh); CPS = 2: half-width tiles, two CTAs per SM
                        auto go_eq = [&](auto VEC, auto CPS, auto WREF) {
                            if constexpr (NC == 1 && C_ == 0) {
                                auto go_ty = [&](auto TYW_) {
                                    constexpr int TYW = TYW_;
                                    using T = EqTile<L, CT, ST, VEC, TYW, CPS>;
                                    auto kern = k_fused_eq<L, CT, ST, VEC, TYW, CPS, (WREF != 0)>;
                                    static int ready[16] = {0};
                                    if (!usable(kern, ready, T::SMEM, (long long)T::REG_PROD * T::NPW * 32 + (long long)T::REG_CONS * T::NCW * 32, T::THREADS)) return;
                                    dim3 g((unsigned)((p.nx + T::TX - 1) / T::TX), (unsigned)((p.ny + TYW - 1) / TYW),
                                           (unsigned)((p.nz + a.i0 - 1) / a.i0));
                                    kern<<<g, T::THREADS, T::SMEM, a.stream>>>(p, a.i0);
                                    if (a.used_kernel) *a.used_kernel = 5;  // LBM_PATH_ONE_PASS_EQ
                                    done = true;
                                };
                                // (7-row tiles where that gives every SM a CTA: full-width tiles, fp64 compute -- plan_fused, a.i2)
                                if constexpr (sizeof(CT) == 8 && CPS == 1) {
                                    if (a.i2 == fs.ty - 1) { go_ty(IC<fs.ty - 1>{}); return; }
                                }
                                go_ty(IC<fs.ty>{});
                            }
                        };
                        // k_fused_eq_split: front / back warps per row (lbm_fused_eq2.cuh); fp32 compute and storage
                        auto go_split = [&](auto EARLY, auto WREF) {
                            constexpr int vec = fused_shape<L, CT, ST, NC>().vec, ty = fused_shape<L, CT, ST, NC>().ty;
                            if constexpr (NC == 1 && C_ == 0 && vec == 4 && sizeof(CT) == 4 && sizeof(ST) == 4) {
                                using T = EqSplitTile<L, CT, ST, vec, ty>;
                                auto kern = k_fused_eq_split<L, CT, ST, vec, ty, (EARLY != 0), (WREF != 0)>;
                                static int ready[16] = {0};
                                if (!usable(kern, ready, T::SMEM, T::REGS_NEEDED, T::THREADS)) return;
                                const int xt = (p.nx + T::TX - 1) / T::TX, yt = (p.ny + ty - 1) / ty, zc = (p.nz + a.i0 - 1) / a.i0;
                                if (a.i1 <= 0) {
                                    kern<<<dim3((unsigned)xt, (unsigned)yt, (unsigned)zc), T::THREADS, T::SMEM, a.stream>>>(p, a.i0, 0, 0);
                                } else {
                                    // one launch per chunk of planes and per group of a.i1 tile rows: every launch is a single
                                    // wave of CTAs that start together (lbm_api.cu, plan_fused)
                                    for (int z = 0; z < zc; ++z)
                                        for (int y0 = 0; y0 < yt; y0 += a.i1)
                                            kern<<<dim3((unsigned)xt, (unsigned)std::min(a.i1, yt - y0), 1u), T::THREADS, T::SMEM, a.stream>>>(p, a.i0, y0, z);
                                }
                                if (a.used_kernel) *a.used_kernel = 5;  // LBM_PATH_ONE_PASS_EQ
                                done = true;
                            }
                        };
                        if (a.eq == 3 || a.eq == 4) {
                            if (a.eq == 4) { if (a.wref) go_split(IC<1>{}, IC<1>{}); else go_split(IC<1>{}, IC<0>{}); }
                            else { if (a.wref) go_split(IC<0>{}, IC<1>{}); else go_split(IC<0>{}, IC<0>{}); }
                            if (!done) {   // not built for this dtype combination: the single-warp row pipeline
                                if (a.wref) go_eq(IC<fs.vec>{}, IC<1>{}, IC<1>{});
                                else go_eq(IC<fs.vec>{}, IC<1>{}, IC<0>{});
                            }
                        } else if (a.eq == 2) {
                            if (a.wref) go_eq(IC<fs.vec / 2>{}, IC<2>{}, IC<1>{});
                            else go_eq(IC<fs.vec / 2>{}, IC<2>{}, IC<0>{});
                        } else if (a.eq == 1) {
                            if (a.wref) go_eq(IC<fs.vec>{}, IC<1>{}, IC<1>{});
                            else go_eq(IC<fs.vec>{}, IC<1>{}, IC<0>{});
                        }
                        if (done) return;
                        if (a.wref) go_ws(IC<1>{});
                        else go_ws(IC<0>{});
                    }
                });
            });
            if (!done) return cudaErrorInvalidValue;
            break;
        }
        default:
            return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}
#endif

}  // namespace lbmk
