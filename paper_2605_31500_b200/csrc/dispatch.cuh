// dispatch.cuh - picks the (dtype, lane-group width, vectors per lane) instantiation of a pass.
#pragma once
#include "internal.h"
#include "kernels.cuh"

namespace gnn {

template <template <typename, int, int> class OpT, Pass PASS, typename Fill>
inline cudaError_t dispatch_pass(int dtype, const Shape& sh, const LaunchCtx& c, Fill fill) {
    auto go = [&](auto* tag) -> cudaError_t {
        using Op = typename std::remove_pointer<decltype(tag)>::type;
        static_assert(Op::NA == kPassInfo[PASS].na && Op::NS == kPassInfo[PASS].ns &&
                          (int)Op::SOFTMAX == kPassInfo[PASS].softmax && (int)Op::HAS_DA == kPassInfo[PASS].has_da,
                      "kPassInfo out of sync with the Op");
        typename Op::Params p;
        fill(p);
        return run_op<Op>(p, sh, c);
    };
    const int gw = group_width(sh.rowv);
    const int nv = sh.rowv > 32 ? 2 : 1;
#define GNN_GO(T)                                                             \
    if (gw == 8) return go((OpT<T, 8, 1>*)nullptr);                           \
    if (gw == 16) return go((OpT<T, 16, 1>*)nullptr);                         \
    if (gw == 32 && nv == 1) return go((OpT<T, 32, 1>*)nullptr);              \
    if (gw == 32 && nv == 2) return go((OpT<T, 32, 2>*)nullptr);
    if (dtype == GNN_F32) { GNN_GO(float) }
    if (dtype == GNN_BF16) { GNN_GO(__nv_bfloat16) }
#undef GNN_GO
    return cudaErrorInvalidValue;
}

}  // namespace gnn
