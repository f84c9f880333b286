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


// Resident warps per SM the register budget is sized for: the carried register rings grow with the number of
// components and reservoirs (DESIGN.md section 5.2 has the count per model).
#if PHX_INST_PREC == 32
#ifndef PHX_MINW_V2
#define PHX_MINW_V2 (PHX_INST_MODEL == 0 ? 16 : 8)   // (reservoir, cfg3: 143.5 Gcell*step/s with the registers of 8 resident warps, 140.7 with 12, 132 with 16)
#endif
#define PHX_MINW_V1 (PHX_INST_MODEL == 0 ? 24 : (PHX_INST_MODEL == 1 ? 20 : 12))
#else
#define PHX_MINW_V2 8
#define PHX_MINW_V1 (PHX_INST_MODEL == 0 ? 16 : (PHX_INST_MODEL == 1 ? 12 : 8))
#endif
#ifndef PHX_MINW_V4
#define PHX_MINW_V4 8
#endif
// The isotropic form (dx == dy): Laplacian as one five-point sum; in the spinor models also bxx == byy, so that the TE-TM
// operator takes Dxx - Dyy in one piece (one packed operation fewer per component and stage).
#define PHX_HAS_ISO 1
// Four cells per lane (two 128-bit loads): complex fp32, scalar model only (the other models run out of registers).
// Two cells per lane in complex fp64 (two 128-bit loads), scalar model only.
#ifndef PHX_HAS_VEC2_64
#define PHX_HAS_VEC2_64 (PHX_INST_PREC == 64 && PHX_INST_MODEL == 0)
#endif
#ifndef PHX_HAS_VEC4
#define PHX_HAS_VEC4 (PHX_INST_PREC == 32 && PHX_INST_MODEL == 0)
#endif

template <int VEC, bool NOISE, bool ZBC, bool ISO, bool DRIVE, bool BULK, bool UNITH = false>
struct Inst {
    static constexpr int MINW = VEC == 4 ? PHX_MINW_V4 : (VEC == 2 ? PHX_MINW_V2 : PHX_MINW_V1);
    static constexpr bool I = ISO && PHX_HAS_ISO;
    // dynamic shared memory: the per-warp rings of the bulk-copy fetch path
    static constexpr size_t SMEM = BULK ? StepSmem<real_t, VEC, PHX_INST_MODEL, DRIVE>::CTA : 0;
    static auto kernel() { return step_kernel<real_t, VEC, PHX_INST_MODEL, NOISE, ZBC, I, DRIVE, MINW, BULK, false, UNITH>; }
    static cudaError_t prepare() {
        if (SMEM > 48 * 1024) {
            static cudaError_t once = cudaFuncSetAttribute(kernel(), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM);
            return once;
        }
        return cudaSuccess;
    }
    static cudaError_t launch(const StepArgs<real_t>& a, dim3 grid, cudaStream_t st) {
        cudaError_t e = prepare();
        if (e != cudaSuccess) return e;
        return launch_maybe_pdl(kernel(), a, grid, SMEM, st);
    }
    static int occupancy() {   // resident CTAs of PHX_STEP_WARPS warps per SM (the register file bounds the WARPS)
        int nb = 0;
        if (prepare() != cudaSuccess ||
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, kernel(), 32 * PHX_STEP_WARPS, SMEM) != cudaSuccess) {
            cudaGetLastError();
            return MINW / PHX_STEP_WARPS;
        }
        return nb;
    }
};

// (the bulk-copy fetch path exists for periodic boundaries; a grid with a zero boundary takes the register loads)
// unith: hbar == 1 exactly; instantiated for the isotropic periodic kernels without drive (the BASELINE grids), the others
// multiply by 1.0f -- the same bits.
template <int VEC, bool NOISE, bool DRIVE, typename F>
static auto dispatch2(bool zbc, bool iso, bool bulk, bool unith, F f) {
    if (zbc) return iso ? f(Inst<VEC, NOISE, true, true, DRIVE, false>()) : f(Inst<VEC, NOISE, true, false, DRIVE, false>());
    if (bulk) return iso ? f(Inst<VEC, NOISE, false, true, DRIVE, true>()) : f(Inst<VEC, NOISE, false, false, DRIVE, true>());
    if constexpr (!DRIVE) {
        if (unith && iso) return f(Inst<VEC, NOISE, false, true, false, false, true>());
    }
    return iso ? f(Inst<VEC, NOISE, false, true, DRIVE, false>()) : f(Inst<VEC, NOISE, false, false, DRIVE, false>());
}

template <int VEC, typename F>
static auto dispatch(bool noise, bool zbc, bool iso, bool drive, bool bulk, bool unith, F f) {
    if (noise && drive) return dispatch2<VEC, true, true>(zbc, iso, bulk, unith, f);   // Eq. (16) carries E and dW together
    if (noise) return dispatch2<VEC, true, false>(zbc, iso, bulk, unith, f);
    if (drive) return dispatch2<VEC, false, true>(zbc, iso, bulk, unith, f);
    return dispatch2<VEC, false, false>(zbc, iso, bulk, unith, f);
}

template <int VEC>
static int occ_vec(bool noise, bool zbc, bool iso, bool drive, bool bulk) {
    return dispatch<VEC>(noise, zbc, iso, drive, bulk, false, [](auto inst) { return decltype(inst)::occupancy(); });
}

template <int VEC>
static cudaError_t launch_vec(const StepArgs<real_t>& a, bool noise, bool zbc, bool iso, bool bulk, dim3 grid, cudaStream_t st) {
    return dispatch<VEC>(noise, zbc, iso, a.E != nullptr, bulk, a.k.ih == real_t(1), [&](auto inst) { return decltype(inst)::launch(a, grid, st); });
}

#define PHX_CAT3(a, b, c) a##b##_##c
#define PHX_NAME(p, m) PHX_CAT3(launch_step_, p, m)

cudaError_t PHX_NAME(PHX_INST_PREC, PHX_INST_MODEL)(const StepArgs<real_t>& a, bool noise, bool zbc, bool iso, bool bulk, int vec,
                                                    dim3 grid, cudaStream_t st) {
#if PHX_INST_PREC == 32
#if PHX_HAS_VEC4
    if (vec == 4) return launch_vec<4>(a, noise, zbc, iso, bulk, grid, st);
#endif
    if (vec == 2) return launch_vec<2>(a, noise, zbc, iso, bulk, grid, st);
#elif PHX_HAS_VEC2_64
    if (vec == 2) return launch_vec<2>(a, noise, zbc, iso, bulk, grid, st);
#endif
    if (vec == 1) return launch_vec<1>(a, noise, zbc, iso, bulk, grid, st);
    return cudaErrorInvalidValue;
}

#define PHX_OCC_NAME(p, m) PHX_CAT3(occupancy_step_, p, m)

// Resident CTAs per SM of the instantiation (for the launch plan: one balanced wave).
int PHX_OCC_NAME(PHX_INST_PREC, PHX_INST_MODEL)(bool noise, bool zbc, bool iso, bool drive, bool bulk, int vec) {
#if PHX_INST_PREC == 32
#if PHX_HAS_VEC4
    if (vec == 4) return occ_vec<4>(noise, zbc, iso, drive, bulk);
#endif
    if (vec == 2) return occ_vec<2>(noise, zbc, iso, drive, bulk);
#elif PHX_HAS_VEC2_64
    if (vec == 2) return occ_vec<2>(noise, zbc, iso, drive, bulk);
#endif
    return occ_vec<1>(noise, zbc, iso, drive, bulk);
}

}  // namespace phx
