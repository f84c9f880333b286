// phx_stepx_inst.cu -- explicit instantiations of the fused step with EXCHANGING STRIPS (phx_step.cuh, template switch XCH)
// for one (precision, model) pair, model 0 (scalar) or 1 (reservoir).  Compiled with -DPHX_INST_PREC={32,64} -DPHX_INST_MODEL={0,1}.
#include "phx_step.cuh"
#include "phx_launch.h"

#ifndef PHX_INST_PREC
#error "compile with -DPHX_INST_PREC=32|64 -DPHX_INST_MODEL=0|1"
#endif

namespace phx {

#if PHX_INST_PREC == 32
typedef float real_t;
#else
typedef double real_t;
#endif

// a.pdl: programmatic stream serialisation (the grid may be scheduled before the previous kernel of the stream has finished; it
// waits in griddepcontrol.wait, phx_step.cuh)
template <typename K>
static cudaError_t launch_maybe_pdl(K kernel, const StepArgs<real_t>& a, dim3 grid, size_t smem, cudaStream_t st) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = dim3(32 * a.wpc);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = a.pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kernel, a);
}


// The exchanging strips of the reservoir model in complex fp32 (cfg5) fetch their rows through the cp.async ring of
// phx_step.cuh (PHX_XCH_RING; the ring is per warp, the CTA has a.wpc of them).
template <int VEC, bool NOISE, bool ISO>
struct InstX {
    static constexpr bool RINGED = step_xch_ringed(PHX_INST_PREC == 64, PHX_INST_MODEL, VEC);
    using SM = StepSmem<real_t, VEC, PHX_INST_MODEL, false>;
    static size_t smem(int warps) { return RINGED ? SM::BARS + (size_t)warps * SM::DEPTH * SM::STAGE : 0; }
    static auto kernel() { return step_kernel<real_t, VEC, PHX_INST_MODEL, NOISE, false, ISO, false, 8, RINGED, true>; }
    static cudaError_t prepare() {
        if (smem(PHX_STEP_XWARPS) > 48 * 1024) {
            static cudaError_t once = cudaFuncSetAttribute(kernel(), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem(PHX_STEP_XWARPS));
            return once;
        }
        return cudaSuccess;
    }
    static cudaError_t launch(const StepArgs<real_t>& a, dim3 grid, cudaStream_t st) {
        cudaError_t e = prepare();
        if (e != cudaSuccess) return e;
        return launch_maybe_pdl(kernel(), a, grid, smem(a.wpc), st);
    }
    static int occupancy(int warps) {
        int nb = 0;
        if (prepare() != cudaSuccess ||
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, kernel(), 32 * warps, smem(warps)) != cudaSuccess) {
            cudaGetLastError();
            return 1;
        }
        return nb;
    }
};

template <int VEC, typename F>
static auto dispatchx(bool noise, bool iso, F f) {
    if (noise) return iso ? f(InstX<VEC, true, true>()) : f(InstX<VEC, true, false>());
    return iso ? f(InstX<VEC, false, true>()) : f(InstX<VEC, false, false>());
}

#if PHX_INST_PREC == 32
#define PHX_XVEC_A 2
#define PHX_XVEC_B 4
#else
#define PHX_XVEC_A 1
#define PHX_XVEC_B 2
#endif

#define PHX_CAT3(a, b, c) a##b##_##c
#define PHX_NAME(p, m) PHX_CAT3(launch_stepx_, p, m)
#define PHX_OCC_NAME(p, m) PHX_CAT3(occupancy_stepx_, p, m)

cudaError_t PHX_NAME(PHX_INST_PREC, PHX_INST_MODEL)(const StepArgs<real_t>& a, bool noise, bool iso, int vec, dim3 grid, cudaStream_t st) {
    if (a.wpc < 1 || a.wpc > PHX_STEP_XWARPS || a.E != nullptr) return cudaErrorInvalidValue;
    if (vec == PHX_XVEC_A) return dispatchx<PHX_XVEC_A>(noise, iso, [&](auto inst) { return decltype(inst)::launch(a, grid, st); });
#if PHX_INST_MODEL == 0
    if (vec == PHX_XVEC_B) return dispatchx<PHX_XVEC_B>(noise, iso, [&](auto inst) { return decltype(inst)::launch(a, grid, st); });
#endif
    return cudaErrorInvalidValue;
}

int PHX_OCC_NAME(PHX_INST_PREC, PHX_INST_MODEL)(bool noise, bool iso, int vec, int warps) {
    if (vec == PHX_XVEC_A) return dispatchx<PHX_XVEC_A>(noise, iso, [&](auto inst) { return decltype(inst)::occupancy(warps); });
#if PHX_INST_MODEL == 0
    if (vec == PHX_XVEC_B) return dispatchx<PHX_XVEC_B>(noise, iso, [&](auto inst) { return decltype(inst)::occupancy(warps); });
#endif
    return 1;
}

}  // namespace phx
