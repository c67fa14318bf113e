// gg_inst_stream2.cu -- the compiled builds of gg_step_stream2 (its own translation unit: gg_inst.h).
#include "gg_stream2.cuh"
#include "gg_inst.h"

namespace gg {
namespace {
template <typename T, int RB, int N0, int N1>
const void* stream2_nw(int nw) {
    switch (nw) {
        case 1: return (const void*)gg_step_stream2<T, RB, N0, N1, 1>;
        case 2: return (const void*)gg_step_stream2<T, RB, N0, N1, 2>;
        case 4: return (const void*)gg_step_stream2<T, RB, N0, N1, 4>;
    }
    return nullptr;
}
template <typename T>
const void* stream2_of(int v, int nw) {
    switch (v) {
        case 0: return stream2_nw<T, 4, 2, 2>(nw);
        case 1: return stream2_nw<T, 3, 2, 2>(nw);
    }
    return nullptr;
}
}  // namespace
const void* stream2_kernel(bool f64, int v, int nw) { return f64 ? stream2_of<double>(v, nw) : stream2_of<float>(v, nw); }
}  // namespace gg
