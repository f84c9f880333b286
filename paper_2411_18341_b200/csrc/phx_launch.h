// phx_launch.h -- host-side entry points of the kernel translation units (internal to libphx).
#pragma once

#include "phx_common.cuh"

// Most warps per CTA of variant STEP (the warps of a CTA are independent: adjacent strips, no barrier between them; the
// launch plan takes 1 or PHX_STEP_WARPS per CTA, whichever leaves fewer warp slots idle: StepArgs::wpc).
#ifndef PHX_STEP_WARPS
#define PHX_STEP_WARPS 2
#endif

// Variant STEP: row iterations a fetch leads its first use by, and the ring length / unroll factor of the row loop.
// (LEAD = 2 costs registers and is slower everywhere: 200.6 against 207.5 Gcell*step/s at 4096^2 fp32, spills in the spinor.)
#ifndef PHX_STEP_LEAD
#define PHX_STEP_LEAD 1
#endif
#define PHX_STEP_RING (4 + PHX_STEP_LEAD)
// Bulk-copy fetch path of variant STEP: stages of the per-warp shared-memory ring (rows in flight = DEPTH - 1); power of 2.
#ifndef PHX_STEP_DEPTH
#define PHX_STEP_DEPTH 8
#endif

namespace phx {

template <typename T> struct StageArgs;

#define PHX_DECL_STAGE(P, T)                                                                                              \
    cudaError_t launch_stage_##P##_0(const StageArgs<T>&, int stage, bool noise, int vec, dim3 grid, dim3 block, cudaStream_t); \
    cudaError_t launch_stage_##P##_1(const StageArgs<T>&, int stage, bool noise, int vec, dim3 grid, dim3 block, cudaStream_t); \
    cudaError_t launch_stage_##P##_2(const StageArgs<T>&, int stage, bool noise, int vec, dim3 grid, dim3 block, cudaStream_t); \
    cudaError_t launch_stage_##P##_3(const StageArgs<T>&, int stage, bool noise, int vec, dim3 grid, dim3 block, cudaStream_t);
PHX_DECL_STAGE(32, float)
PHX_DECL_STAGE(64, double)
#undef PHX_DECL_STAGE

template <typename T> struct StepArgs;

#define PHX_DECL_STEP(P, T)                                                                                      \
    cudaError_t launch_step_##P##_0(const StepArgs<T>&, bool noise, bool zbc, bool iso, bool bulk, int vec, dim3 grid, cudaStream_t); \
    cudaError_t launch_step_##P##_1(const StepArgs<T>&, bool noise, bool zbc, bool iso, bool bulk, int vec, dim3 grid, cudaStream_t); \
    cudaError_t launch_step_##P##_2(const StepArgs<T>&, bool noise, bool zbc, bool iso, bool bulk, int vec, dim3 grid, cudaStream_t); \
    cudaError_t launch_step_##P##_3(const StepArgs<T>&, bool noise, bool zbc, bool iso, bool bulk, int vec, dim3 grid, cudaStream_t); \
    int occupancy_step_##P##_0(bool noise, bool zbc, bool iso, bool drive, bool bulk, int vec);                                          \
    int occupancy_step_##P##_1(bool noise, bool zbc, bool iso, bool drive, bool bulk, int vec);                                          \
    int occupancy_step_##P##_2(bool noise, bool zbc, bool iso, bool drive, bool bulk, int vec);                                          \
    int occupancy_step_##P##_3(bool noise, bool zbc, bool iso, bool drive, bool bulk, int vec);
PHX_DECL_STEP(32, float)
PHX_DECL_STEP(64, double)
#undef PHX_DECL_STEP

// phx_resident.cu: variant RESIDENT (a small grid on chip for all steps of one launch)
#ifndef PHX_RESIDENT_THREADS
#define PHX_RESIDENT_THREADS 512
#endif
template <typename T>
struct ResidentArgs {
    Geom geo;
    Coef<T> k;
    typename Cx<T>::type* psi;      // state [batch][ny][nx], advanced in place
    T* n;                           // reservoir state, or nullptr
    const T* V;                     // [ny][nx] or nullptr
    const T* P;                     // [ny][nx] or nullptr
    uint64_t* step_slots;           // both device step-counter slots receive step0 + n_steps
    uint64_t step0;                 // completed steps before this launch
    int n_steps;
    uint32_t seed;
};
int resident_cpt(size_t cells, int prec64, bool res);     // cells per thread, 0 = the grid does not fit
cudaError_t launch_resident_32(const ResidentArgs<float>&, bool res, bool noise, cudaStream_t);
cudaError_t launch_resident_64(const ResidentArgs<double>&, bool res, bool noise, cudaStream_t);

// phx_aux.cu: small helper kernels
cudaError_t launch_ensemble_mean(const void* psi, void* out, int prec64, size_t plane, int batch, cudaStream_t);
cudaError_t launch_noise_words(uint32_t* out, uint32_t seed, uint64_t step, size_t plane, int r0, int batch, cudaStream_t);

}  // namespace phx
