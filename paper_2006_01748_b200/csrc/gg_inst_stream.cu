// gg_inst_stream.cu -- the compiled builds of gg_step_stream (its own translation unit: gg_inst.h).
#include "gg_stream.cuh"
#include "gg_inst.h"

namespace gg {
namespace {
template <typename T, int RB, int NST>
const void* stream_nw(int nw) {
    switch (nw) {
        case 1: return (const void*)gg_step_stream<T, RB, NST, 1>;
        case 2: return (const void*)gg_step_stream<T, RB, NST, 2>;
        case 4: return (const void*)gg_step_stream<T, RB, NST, 4>;
        case 8: return (const void*)gg_step_stream<T, RB, NST, 8>;
    }
    return nullptr;
}
template <typename T>
const void* stream_of(int v, int nw) {
    switch (v) {
        case 0: return stream_nw<T, 2, 4>(nw);
        case 1: return stream_nw<T, 4, 2>(nw);
    }
    return nullptr;
}
}  // namespace
const void* stream_kernel(bool f64, int v, int nw) { return f64 ? stream_of<double>(v, nw) : stream_of<float>(v, nw); }
}  // namespace gg
