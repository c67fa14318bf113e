// gg_inst.h -- where the compiled builds of the step kernels live.
// Each family of builds is instantiated in its own translation unit (gg_inst_*.cu), so that nvcc
// compiles the families in parallel (paper_2006_01748_b200/build.py: --threads); gg_api.cu only
// looks their addresses up through these host functions.  nullptr = no such build.
#pragma once

namespace gg {

// GG_KERNEL_QUAD, build v of gg_pair_plan.inc: kQuadVariants (rows per stage, ring0 stages, ring1
// stages, coefficient-ring stages, warps per role)
const void* quad_kernel(bool f64, int v);
// GG_KERNEL_PAIR, build v of kPairVariants (rows per stage, stages)
const void* pair_kernel(bool f64, int v);
// GG_KERNEL_STREAM, build v of kVariants (rows per box, stages) with nw in {1, 2, 4, 8} warps per CTA
const void* stream_kernel(bool f64, int v, int nw);
// GG_KERNEL_STREAM2, build v of kVariants2 (rows per box, ring0 stages, ring1 stages), nw in {1, 2, 4}
const void* stream2_kernel(bool f64, int v, int nw);

}  // namespace gg
