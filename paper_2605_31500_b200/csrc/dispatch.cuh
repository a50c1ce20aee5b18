// dispatch.cuh - picks the (dtype, bytes per lane, lane-group width) instantiation of a pass.
#pragma once
#include "internal.h"
#include "kernels.cuh"

namespace gnn {

template <template <typename, int, int, int> class OpT, Pass PASS, typename Fill>
inline cudaError_t dispatch_pass(int dtype, const Shape& sh0, const LaunchCtx& c, Fill fill) {
    LaneCfg lc;
    const Shape sh = pass_shape(sh0, PASS, dtype == GNN_F32 ? 4 : 2, lc);
    auto go = [&](auto* tag) -> cudaError_t {
        using Op = typename std::remove_pointer<decltype(tag)>::type;
        static_assert(Op::NA == kPassInfo[PASS].na && Op::NS == kPassInfo[PASS].ns &&
                          (int)Op::SOFTMAX == kPassInfo[PASS].softmax && (int)Op::HAS_DA == kPassInfo[PASS].has_da,
                      "kPassInfo out of sync with the Op");
        typename Op::Params p;
        fill(p);
        return run_op<Op>(p, sh, c);
    };
#define GNN_G(T, CB)                                                                         \
    {                                                                                        \
        constexpr int KU = pass_ku(PASS, CB); /* edges per batch; never more than the group width */ \
        if (lc.g == 4) return go((OpT<T, CB, 4, (KU < 4 ? KU : 4)>*)nullptr);                \
        if (lc.g == 8) return go((OpT<T, CB, 8, (KU < 8 ? KU : 8)>*)nullptr);                \
        if (lc.g == 16) return go((OpT<T, CB, 16, KU>*)nullptr);                             \
        if (lc.g == 32) return go((OpT<T, CB, 32, KU>*)nullptr);                             \
    }
#define GNN_GO(T)                                                                            \
    if (lc.cb == 16) GNN_G(T, 16)                                                            \
    if (lc.cb == 32) GNN_G(T, 32)
    if (dtype == GNN_F32) { GNN_GO(float) }
    if (dtype == GNN_BF16) { GNN_GO(__nv_bfloat16) }
#undef GNN_GO
#undef GNN_G
    return cudaErrorInvalidValue;
}

}  // namespace gnn
