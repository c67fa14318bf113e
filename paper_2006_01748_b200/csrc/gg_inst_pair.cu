// gg_inst_pair.cu -- the compiled builds of gg_step_pair (its own translation unit: gg_inst.h).
#include "gg_pair.cuh"
#include "gg_inst.h"

namespace gg {
namespace {
template <typename T>
const void* pair_of(int v) {
    switch (v) {
        case 0: return (const void*)gg_step_pair<T, 4, 2>;
        case 1: return (const void*)gg_step_pair<T, 3, 3>;
    }
    return nullptr;
}
}  // namespace
const void* pair_kernel(bool f64, int v) { return f64 ? pair_of<double>(v) : pair_of<float>(v); }
}  // namespace gg
