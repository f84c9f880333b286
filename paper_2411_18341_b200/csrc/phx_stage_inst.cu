// phx_stage_inst.cu -- explicit instantiations of the per-stage kernels for one (precision, model) pair.
// Compiled once per pair with -DPHX_INST_PREC={32,64} -DPHX_INST_MODEL={0..3} so the pairs build in parallel.
#include "phx_stage.cuh"
#include "phx_launch.h"

#ifndef PHX_INST_PREC
#error "compile with -DPHX_INST_PREC=32|64 -DPHX_INST_MODEL=0..3"
#endif

namespace phx {

#if PHX_INST_PREC == 32
typedef float real_t;
#else
typedef double real_t;
#endif

template <int VEC, int STAGE, bool NOISE>
static cudaError_t launch_one(const StageArgs<real_t>& a, dim3 grid, dim3 block, cudaStream_t st) {
    stage_kernel<real_t, VEC, PHX_INST_MODEL, STAGE, NOISE><<<grid, block, 0, st>>>(a);
    return cudaGetLastError();
}

template <int VEC>
static cudaError_t launch_vec(const StageArgs<real_t>& a, int stage, bool noise, dim3 grid, dim3 block, cudaStream_t st) {
    switch (stage) {
        case 1: return launch_one<VEC, 1, false>(a, grid, block, st);
        case 2: return launch_one<VEC, 2, false>(a, grid, block, st);
        case 3: return launch_one<VEC, 3, false>(a, grid, block, st);
        case 4: return noise ? launch_one<VEC, 4, true>(a, grid, block, st) : launch_one<VEC, 4, false>(a, grid, block, st);
    }
    return cudaErrorInvalidValue;
}

#define PHX_CAT3(a, b, c) a##b##_##c
#define PHX_NAME(p, m) PHX_CAT3(launch_stage_, p, m)

cudaError_t PHX_NAME(PHX_INST_PREC, PHX_INST_MODEL)(const StageArgs<real_t>& a, int stage, bool noise, int vec, dim3 grid,
                                                    dim3 block, cudaStream_t st) {
    if (vec == 2) return launch_vec<2>(a, stage, noise, grid, block, st);
    return launch_vec<1>(a, stage, noise, grid, block, st);
}

}  // namespace phx
