// gg_inst_quad.cu -- the compiled builds of gg_step_quad (its own translation unit: gg_inst.h).
#include "gg_quad.cuh"
#include "gg_inst.h"

namespace gg {
namespace {
template <typename T>
const void* quad_of(int v) {
    switch (v) {
        case 0: return (const void*)gg_step_quad<T, 4, 2, 2, 0, 4>;
        case 1: return (const void*)gg_step_quad<T, 4, 2, 2, 2, 4>;
        case 2: return (const void*)gg_step_quad<T, 4, 2, 2, 2, 2>;
    }
    return nullptr;
}
}  // namespace
const void* quad_kernel(bool f64, int v) { return f64 ? quad_of<double>(v) : quad_of<float>(v); }
}  // namespace gg
