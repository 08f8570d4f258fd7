// lbm_launch.cuh -- host-side dispatch from run-time options to the kernel templates of lbm_core.cuh.
// One translation unit per (lattice, compute dtype, storage dtype) instantiates launch<L,CT,ST>.
#pragma once
#include "lbm_hot.cuh"

namespace lbmk {

enum Op { OP_MOMENTS = 0, OP_VIRTUAL = 1, OP_STEP = 2, OP_INIT = 3, OP_EXPORT_MACRO = 4, OP_EXPORT_POP = 5, OP_IMPORT_POP = 6, OP_UNSTREAM = 7 };

struct LaunchArgs {
    int op;
    int nc;    // components
    int coll;  // 0 BGK, 1 MRT, 2 none (pure streaming)
    int vec;   // cells per thread along x in the hot kernels: 1 or vec_width<CT, ST, NC>() (needs nx % vec == 0)
    int bnd;   // any solid cell or non-periodic axis
    const void* params;  // KParams<CT>
    const void* a0;      // op-specific (FieldIO<CT>* for init / import / export_pop; u_out for export_macro)
    const void* a1;
    void* a2;
    int i0;
    cudaStream_t stream;
};

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
    switch (a.op) {
        case OP_MOMENTS:
            with_nc([&](auto NC) {
                with_bnd([&](auto B) {
                    constexpr int VW = vec_width<CT, ST, NC>();
                    if (a.vec == VW && VW > 1)
                        k_moments_v<L, NC, CT, ST, (B != 0), VW><<<grid(p.N / VW, 256), 256, 0, a.stream>>>(p);
                    else
                        k_moments_v<L, NC, CT, ST, (B != 0), 1><<<grid(p.N, 256), 256, 0, a.stream>>>(p);
                });
            });
            break;
        case OP_VIRTUAL:
            if (p.nbsolid > 0)
                with_nc([&](auto NC) { k_virtual_density<L, NC, CT><<<grid(p.nbsolid, 128), 128, 0, a.stream>>>(p); });
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
                        if (a.vec == VW && VW > 1)
                            k_step_v<L, NC, CT, ST, C_, (B != 0), VW><<<grid(p.N / VW, 128), 128, 0, a.stream>>>(p);
                        else
                            k_step_v<L, NC, CT, ST, C_, (B != 0), 1><<<grid(p.N, 128), 128, 0, a.stream>>>(p);
                    });
                });
            });
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
        default:
            return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}
#endif

}  // namespace lbmk
