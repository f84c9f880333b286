// phx_step_inst.cu -- explicit instantiations of the fused-step kernels (variant STEP) for one (precision, model)
// pair.  Compiled once per pair with -DPHX_INST_PREC={32,64} -DPHX_INST_MODEL={0..3} so the pairs build in parallel.
#include "phx_step.cuh"
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

// Resident CTAs (of 4 warps) per SM the register budget is sized for: the carried register windows grow with the
// number of components and reservoirs (DESIGN.md section 5.2 has the count per model).
#if PHX_INST_PREC == 32
#ifndef PHX_MINB_V2
#define PHX_MINB_V2 (PHX_INST_MODEL == 0 ? 4 : (PHX_INST_MODEL == 1 ? 3 : 2))
#endif
#define PHX_MINB_V1 (PHX_INST_MODEL == 0 ? 6 : (PHX_INST_MODEL == 1 ? 5 : 3))
#else
#define PHX_MINB_V2 2
#define PHX_MINB_V1 (PHX_INST_MODEL == 0 ? 4 : (PHX_INST_MODEL == 1 ? 3 : 2))
#endif

template <int VEC, bool NOISE, bool ZBC>
static cudaError_t launch_one(const StepArgs<real_t>& a, dim3 grid, cudaStream_t st) {
    constexpr int MINB = VEC == 2 ? PHX_MINB_V2 : PHX_MINB_V1;
    step_kernel<real_t, VEC, PHX_INST_MODEL, NOISE, ZBC, MINB><<<grid, 128, 0, st>>>(a);
    return cudaGetLastError();
}

template <int VEC, bool NOISE, bool ZBC>
static int occ_one() {
    constexpr int MINB = VEC == 2 ? PHX_MINB_V2 : PHX_MINB_V1;
    int nb = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, step_kernel<real_t, VEC, PHX_INST_MODEL, NOISE, ZBC, MINB>, 128, 0) != cudaSuccess) {
        cudaGetLastError();
        return MINB;
    }
    return nb;
}

template <int VEC>
static int occ_vec(bool noise, bool zbc) {
    if (noise) return zbc ? occ_one<VEC, true, true>() : occ_one<VEC, true, false>();
    return zbc ? occ_one<VEC, false, true>() : occ_one<VEC, false, false>();
}

template <int VEC>
static cudaError_t launch_vec(const StepArgs<real_t>& a, bool noise, bool zbc, dim3 grid, cudaStream_t st) {
    if (noise) return zbc ? launch_one<VEC, true, true>(a, grid, st) : launch_one<VEC, true, false>(a, grid, st);
    return zbc ? launch_one<VEC, false, true>(a, grid, st) : launch_one<VEC, false, false>(a, grid, st);
}

#define PHX_CAT3(a, b, c) a##b##_##c
#define PHX_NAME(p, m) PHX_CAT3(launch_step_, p, m)

cudaError_t PHX_NAME(PHX_INST_PREC, PHX_INST_MODEL)(const StepArgs<real_t>& a, bool noise, bool zbc, int vec, dim3 grid,
                                                    cudaStream_t st) {
#if PHX_INST_PREC == 32
    if (vec == 2) return launch_vec<2>(a, noise, zbc, grid, st);
#endif
    if (vec == 1) return launch_vec<1>(a, noise, zbc, grid, st);
    return cudaErrorInvalidValue;
}

#define PHX_OCC_NAME(p, m) PHX_CAT3(occupancy_step_, p, m)

// Resident CTAs per SM of the instantiation (for the launch plan: one balanced wave).
int PHX_OCC_NAME(PHX_INST_PREC, PHX_INST_MODEL)(bool noise, bool zbc, int vec) {
#if PHX_INST_PREC == 32
    if (vec == 2) return occ_vec<2>(noise, zbc);
#endif
    return occ_vec<1>(noise, zbc);
}

}  // namespace phx
