// phx_step.cuh -- variant STEP: one kernel per RK4 step, the four stages temporally blocked on chip
// (DESIGN.md section 5.2).  The idea is the paper's subgrid decomposition with N_halo = 4 (PAPER.md:167-173,
// :183: a whole time step on a haloed subgrid is independent of its neighbours), re-designed for B200:
// the "subgrid" is a warp-wide column strip that streams down y, and the haloed data live in REGISTERS.
//
// One warp owns a strip of W = 32*VEC columns (VEC cells per lane, one 128-bit load for complex fp32 pairs)
// of which the inner W-8 are output columns, and walks a chunk of rows.  The four stages run as a software
// pipeline along y: in the iteration whose front row is j,
//     stage 1 evaluates K1 on row j   from psi rows j-1..j+1  -> y2[j]   = psi + dt/2 K1, acc  = psi + dt/6 K1
//     stage 2 evaluates K2 on row j-1 from y2  rows j-2..j    -> y3[j-1] = psi + dt/2 K2, acc += dt/3 K2
//     stage 3 evaluates K3 on row j-2 from y3  rows j-3..j-1  -> y4[j-2] = psi + dt   K3, acc += dt/3 K3
//     stage 4 evaluates K4 on row j-3 from y4  rows j-4..j-2  -> psi(t+dt)[j-3] = acc + dt/6 K4 (+ dW, Eq. (22))
// (Eqs. (2)-(6)).  Every stage input is a three-row register window per lane; x neighbours
// come from warp shuffles, so there is no shared memory and no block-level barrier.  The four halo columns
// on each side of the strip are recomputed redundantly (their lanes compute values that are never stored;
// each stage invalidates one more column from either edge), the 4+4 halo rows of a chunk likewise.
// HBM traffic per cell-step: read psi, V once, write psi once (+ halo re-reads, mostly L2 hits) instead of the
// 14 complex transfers of variant STAGE.  psi(t) and psi(t+dt) are distinct buffers (ping-pong).
#pragma once

#include <climits>

#include "phx_common.cuh"
#include "phx_deriv.cuh"
#include "phx_philox.cuh"
#include "phx_launch.h"

#ifndef PHX_STEP_PF_ROWS
#define PHX_STEP_PF_ROWS 4
#endif
// Second prefetch level (L2 -> L1) this many row iterations ahead of the register fetch; 0 = none.
// 256-bit global loads / stores of a lane's four complex fp32 cells (sm_100: LDG.E.256) instead of two 128-bit ones.
// Measured: 216.9 against 218.8 Gcell*step/s at 4096^2, equal at 8192^2 (229): off.
#ifndef PHX_STEP_LD256
#define PHX_STEP_LD256 0
#endif
#ifndef PHX_STEP_PF1_ROWS
#define PHX_STEP_PF1_ROWS 0
#endif

namespace phx {

template <typename T>
struct StepArgs {
    using C = typename Cx<T>::type;
    Geom geo;
    Coef<T> k;
    const C* psi_in[2];
    C* psi_out[2];
    const T* n_in[2];
    T* n_out[2];
    const T* V;                 // [ny][nx] or nullptr
    const T* P;                 // [ny][nx] or nullptr
    const C* E;                 // [ny][nx] drive amplitude E(r) (kernels instantiated with DRIVE only)
    const uint64_t* step_in;    // completed steps before this one
    uint64_t* step_out;         // receives step_in + 1 (the slot the next launch reads)
    uint32_t seed;
    int ly;                     // rows per chunk
    int strips;                 // strips per row of the grid
    int wpc;                    // warps per CTA of this launch (1 .. PHX_STEP_WARPS; the warps of a CTA are independent)
    int x0;                     // first output column of strip 0 (0, except in the side launch that covers a ragged last strip)
    int pdl;                    // (host side) launch as a programmatic dependent of the previous kernel of the stream
};

namespace stepk {

template <int VEC> __device__ __forceinline__ void ldc(const float2* p, float2 (&v)[VEC]) {
#if PHX_STEP_LD256
    if constexpr (VEC == 4) {       // one 256-bit load (sm_100: LDG.E.256); the lane's four cells are 32-byte aligned
        asm volatile("ld.global.nc.v8.f32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                     : "=f"(v[0].x), "=f"(v[0].y), "=f"(v[1].x), "=f"(v[1].y), "=f"(v[2].x), "=f"(v[2].y), "=f"(v[3].x), "=f"(v[3].y) : "l"(p));
    } else
#endif
    if constexpr (VEC % 2 == 0) {
#pragma unroll
        for (int h = 0; h < VEC / 2; ++h) {
            const float4 q = __ldg(reinterpret_cast<const float4*>(p) + h);
            v[2 * h] = make_float2(q.x, q.y);
            v[2 * h + 1] = make_float2(q.z, q.w);
        }
    } else v[0] = __ldg(p);
}
template <int VEC> __device__ __forceinline__ void ldc(const double2* p, double2 (&v)[VEC]) {
#pragma unroll
    for (int i = 0; i < VEC; ++i) v[i] = __ldg(p + i);
}
template <int VEC> __device__ __forceinline__ void stc(float2* p, const float2 (&v)[VEC]) {
#if PHX_STEP_LD256
    if constexpr (VEC == 4) {
        asm volatile("st.global.v8.f32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"l"(p), "f"(v[0].x), "f"(v[0].y), "f"(v[1].x), "f"(v[1].y),
                     "f"(v[2].x), "f"(v[2].y), "f"(v[3].x), "f"(v[3].y) : "memory");
    } else
#endif
    if constexpr (VEC % 2 == 0) {
#pragma unroll
        for (int h = 0; h < VEC / 2; ++h) reinterpret_cast<float4*>(p)[h] = make_float4(v[2 * h].x, v[2 * h].y, v[2 * h + 1].x, v[2 * h + 1].y);
    } else *p = v[0];
}
template <int VEC> __device__ __forceinline__ void stc(double2* p, const double2 (&v)[VEC]) {
#pragma unroll
    for (int i = 0; i < VEC; ++i) p[i] = v[i];
}
template <int VEC> __device__ __forceinline__ void ldr(const float* p, float (&v)[VEC]) {
    if constexpr (VEC == 4) { const float4 q = __ldg(reinterpret_cast<const float4*>(p)); v[0] = q.x; v[1] = q.y; v[2] = q.z; v[3] = q.w; }
    else if constexpr (VEC == 2) { const float2 q = __ldg(reinterpret_cast<const float2*>(p)); v[0] = q.x; v[1] = q.y; }
    else v[0] = __ldg(p);
}
template <int VEC> __device__ __forceinline__ void ldr(const double* p, double (&v)[VEC]) {
    if constexpr (VEC == 2) { const double2 q = __ldg(reinterpret_cast<const double2*>(p)); v[0] = q.x; v[1] = q.y; }
    else v[0] = __ldg(p);
}
template <int VEC> __device__ __forceinline__ void str(float* p, const float (&v)[VEC]) {
    if constexpr (VEC == 4) *reinterpret_cast<float4*>(p) = make_float4(v[0], v[1], v[2], v[3]);
    else if constexpr (VEC == 2) *reinterpret_cast<float2*>(p) = make_float2(v[0], v[1]);
    else *p = v[0];
}
template <int VEC> __device__ __forceinline__ void str(double* p, const double (&v)[VEC]) {
    if constexpr (VEC == 2) *reinterpret_cast<double2*>(p) = make_double2(v[0], v[1]);
    else *p = v[0];
}

// ---- bulk-copy fetch path (template switch BULK): rows are brought from global memory into a per-warp ring of shared-memory
// stages by 1-D bulk copies of the TMA unit (cp.async.bulk, one elected lane, completion on an mbarrier), DEPTH rows ahead
// of their use, and read from there with 128-bit shared loads.  No register is tied up by a row in flight from DRAM. ----
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
// (the issuing instructions are predicated on `lead` -- one elected lane -- instead of sitting in a divergent branch)
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes, uint32_t lead) {
    asm volatile("{\n.reg .pred p;\nsetp.ne.u32 p, %2, 0;\n@p mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n}"
                 ::"r"(bar), "r"(bytes), "r"(lead) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra DONE;\n"
        "bra LAB_WAIT;\n"
        "DONE:\n"
        "}" ::"r"(bar), "r"(parity) : "memory");
}
// non-blocking: has the phase with this parity completed?
__device__ __forceinline__ uint32_t mbar_test(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile("{\n.reg .pred p;\nmbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}"
                 : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok;
}
// global -> shared bulk copy of `bytes` (a multiple of 16; both addresses 16-byte aligned), completing on `bar`
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar, uint32_t lead) {
    asm volatile("{\n.reg .pred p;\nsetp.ne.u32 p, %4, 0;\n"
                 "@p cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n}"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar), "r"(lead) : "memory");
}
// cp.async form of the same ring (step_ring_cpasync, phx_launch.h): every LANE copies its own cells global -> shared with cp.async
// (LDGSTS, 16 / 8 / 4 bytes), one commit group per row iteration, cp.async.wait_group before the row is read back.  A lane
// only ever reads what it copied itself: no mbarrier, no elected lane, no __syncwarp, and a strip that crosses the periodic
// edge needs no second piece (the lane's wrapped column addresses it).
template <int BYTES> __device__ __forceinline__ void cpasync(uint32_t dst, const void* src) {
    if constexpr (BYTES >= 16) {
#pragma unroll
        for (int o = 0; o < BYTES; o += 16)
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst + o), "l"(static_cast<const char*>(src) + o) : "memory");
    } else {
        asm volatile("cp.async.ca.shared.global [%0], [%1], %2;" ::"r"(dst), "l"(src), "n"(BYTES) : "memory");
    }
}

// A lane's complex cells in the cp.async ring.  PHX_RING_PLANE = 16: a lane's 16-byte chunks sit next to each other (lane
// stride 32 bytes when a lane holds 4 cells fp32 / 2 cells fp64).  PHX_RING_PLANE = 512 stores the row as planes of 16-byte
// chunks (chunk h of lane l at row + h * 512 + l * 16) so that the 128-bit shared accesses of a warp are contiguous:
// measured SLOWER (cfg2 4096^2 fp64 91.7 against 102.6-103.3 Gcell*step/s in the same run), so it is off.
#ifndef PHX_RING_PLANE
#define PHX_RING_PLANE 16
#endif
// The cp.async kernels may leave the row loop early like the register-load kernels (measured neutral).
#ifndef PHX_RING_EXIT
#define PHX_RING_EXIT 1
#endif
template <int BYTES> __device__ __forceinline__ void ring_cp(uint32_t row, int lane, const void* src) {
    if constexpr (BYTES > 16) {
#pragma unroll
        for (int h = 0; h < BYTES / 16; ++h)
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(row + h * PHX_RING_PLANE + lane * (PHX_RING_PLANE == 512 ? 16 : BYTES) + (PHX_RING_PLANE == 512 ? 0 : 0)), "l"(static_cast<const char*>(src) + h * 16) : "memory");
    } else cpasync<BYTES>(row + lane * BYTES, src);
}
template <int VEC> __device__ __forceinline__ void ring_ld(const unsigned char* row, int lane, float2 (&v)[VEC]) {
    if constexpr (VEC == 4) {
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const float4 q = *reinterpret_cast<const float4*>(row + h * PHX_RING_PLANE + lane * (PHX_RING_PLANE == 512 ? 16 : 32));
            v[2 * h] = make_float2(q.x, q.y);
            v[2 * h + 1] = make_float2(q.z, q.w);
        }
    } else if constexpr (VEC == 2) {
        const float4 q = *reinterpret_cast<const float4*>(row + lane * 16);
        v[0] = make_float2(q.x, q.y);
        v[1] = make_float2(q.z, q.w);
    } else v[0] = *reinterpret_cast<const float2*>(row + lane * 8);
}
template <int VEC> __device__ __forceinline__ void ring_ld(const unsigned char* row, int lane, double2 (&v)[VEC]) {
#pragma unroll
    for (int h = 0; h < VEC; ++h) v[h] = *reinterpret_cast<const double2*>(row + h * PHX_RING_PLANE + lane * (PHX_RING_PLANE == 512 ? 16 : 16 * VEC));
}

template <int VEC> __device__ __forceinline__ void ldsc(const float2* p, float2 (&v)[VEC]) {
    if constexpr (VEC % 2 == 0) {
#pragma unroll
        for (int h = 0; h < VEC / 2; ++h) {
            const float4 q = reinterpret_cast<const float4*>(p)[h];
            v[2 * h] = make_float2(q.x, q.y);
            v[2 * h + 1] = make_float2(q.z, q.w);
        }
    } else v[0] = *p;
}
template <int VEC> __device__ __forceinline__ void ldsc(const double2* p, double2 (&v)[VEC]) {
#pragma unroll
    for (int i = 0; i < VEC; ++i) v[i] = p[i];
}
template <int VEC> __device__ __forceinline__ void ldsr(const float* p, float (&v)[VEC]) {
    if constexpr (VEC == 4) { const float4 q = *reinterpret_cast<const float4*>(p); v[0] = q.x; v[1] = q.y; v[2] = q.z; v[3] = q.w; }
    else if constexpr (VEC == 2) { const float2 q = *reinterpret_cast<const float2*>(p); v[0] = q.x; v[1] = q.y; }
    else v[0] = *p;
}
template <int VEC> __device__ __forceinline__ void ldsr(const double* p, double (&v)[VEC]) {
    if constexpr (VEC == 2) { const double2 q = *reinterpret_cast<const double2*>(p); v[0] = q.x; v[1] = q.y; }
    else v[0] = *p;
}

// Shared-memory accesses of the exchanging strips: volatile, so that the compiler keeps them in program order; the LSU
// executes the shared-memory instructions of a warp in order, and that is all the ordering the protocol needs (a fence
// here would also wait for the global loads in flight, which the row loop keeps in flight on purpose; measured: 67 against
// 88 Gcell*step/s on cfg5 with __threadfence_block()).  No "memory" clobber: volatile asm statements keep their order among
// themselves, and the global loads and stores of the row loop stay free to move across them.
__device__ __forceinline__ void xst(float2* p, float2 v) { asm volatile("st.volatile.shared.v2.f32 [%0], {%1, %2};" ::"r"(smem_u32(p)), "f"(v.x), "f"(v.y)); }
__device__ __forceinline__ void xst(double2* p, double2 v) { asm volatile("st.volatile.shared.v2.f64 [%0], {%1, %2};" ::"r"(smem_u32(p)), "d"(v.x), "d"(v.y)); }
__device__ __forceinline__ float2 xld(const float2* p) { float2 v; asm volatile("ld.volatile.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(smem_u32(p))); return v; }
__device__ __forceinline__ double2 xld(const double2* p) { double2 v; asm volatile("ld.volatile.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(smem_u32(p))); return v; }
__device__ __forceinline__ void xst_flag(int* p, int v) { asm volatile("st.volatile.shared.s32 [%0], %1;" ::"r"(smem_u32(p)), "r"(v)); }
__device__ __forceinline__ int xld_flag(const int* p) { int v; asm volatile("ld.volatile.shared.s32 %0, [%1];" : "=r"(v) : "r"(smem_u32(p))); return v; }

// DRAM -> L2 prefetch of the line holding p (no register is tied up; the register fetch one row ahead then hits L2).
__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }
__device__ __forceinline__ void prefetch_l1(const void* p) { asm volatile("prefetch.global.L1 [%0];" ::"l"(p)); }

__device__ __forceinline__ float2 up1(float2 v) { return make_float2(__shfl_up_sync(0xffffffffu, v.x, 1), __shfl_up_sync(0xffffffffu, v.y, 1)); }
__device__ __forceinline__ float2 dn1(float2 v) { return make_float2(__shfl_down_sync(0xffffffffu, v.x, 1), __shfl_down_sync(0xffffffffu, v.y, 1)); }
__device__ __forceinline__ double2 up1(double2 v) { return make_double2(__shfl_up_sync(0xffffffffu, v.x, 1), __shfl_up_sync(0xffffffffu, v.y, 1)); }
__device__ __forceinline__ double2 dn1(double2 v) { return make_double2(__shfl_down_sync(0xffffffffu, v.x, 1), __shfl_down_sync(0xffffffffu, v.y, 1)); }

// Neighbourhood of cell i of the centre row (rc) of a three-row window (rs = row below, rn = row above);
// west/east of the lane's cells by shuffle.  NINE (spinor models): the corner difference Dxy4 is formed from the
// vertical differences n - s of the neighbouring columns, so that one pair per side crosses lanes instead of two.
// XCH (the warps of a CTA tile the whole row, see step_kernel): lane 0 takes its west neighbour and lane 31 its east
// neighbour from `edge`, the cell the neighbouring warp published in shared memory.
template <typename T, int VEC, bool NINE, bool XCH = false>
__device__ __forceinline__ void gather(const typename Cx<T>::type (&rs)[VEC], const typename Cx<T>::type (&rc)[VEC],
                                       const typename Cx<T>::type (&rn)[VEC], Nbhd<T> (&nb)[VEC], int lane = 0,
                                       typename Cx<T>::type edge = typename Cx<T>::type()) {
    using C = typename Cx<T>::type;
    C west = up1(rc[VEC - 1]);
    C east = dn1(rc[0]);
    if (XCH) {          // edge: read from shared memory at the top of the iteration (one load per lane: lane 0 the last cell of the
        // strip to the west, lane 31 the first of the strip to the east) and selected in here.  Loading it here, next to its use,
        // measured 94 against 105 Gcell*step/s on cfg5; a predicated load straight into the shuffled register (no select) 97.
        if (lane == 0) west = edge;
        if (lane == 31) east = edge;
    }
#pragma unroll
    for (int i = 0; i < VEC; ++i) {
        nb[i].c = rc[i];
        nb[i].s = rs[i];
        nb[i].n = rn[i];
        nb[i].w = i == 0 ? west : rc[i - 1];
        nb[i].e = i == VEC - 1 ? east : rc[i + 1];
    }
    if (NINE) {
        C vd[VEC];
#pragma unroll
        for (int i = 0; i < VEC; ++i) vd[i] = sub2(rn[i], rs[i]);
        const C vwest = up1(vd[VEC - 1]);
        const C veast = dn1(vd[0]);
#pragma unroll
        for (int i = 0; i < VEC; ++i) nb[i].D = sub2(i == VEC - 1 ? veast : vd[i + 1], i == 0 ? vwest : vd[i - 1]);
    }
}

}  // namespace stepk

// Rows carried in registers live in RINGS of PHX_STEP_RING slots: the row with number q sits in slot q mod RING of
// its ring for as long as it is live, and the row loop is unrolled RING times, so that every slot index is a
// compile-time constant and moving the windows down by one row costs no instruction (a dead slot costs no
// register either).  RING = 4 + LEAD is the longest life: psi rows j-2 .. j+1+LEAD and V rows j-3 .. j+LEAD, where LEAD
// (PHX_STEP_LEAD, phx_launch.h) is the number of row iterations a fetch leads its first use by.

// Byte layout of the per-warp shared-memory ring of the bulk-copy fetch path: PHX_STEP_DEPTH stages, each holding what one
// row iteration fetches for the warp's strip of W columns: psi row j+1+LEAD of every component, then the row-local inputs
// (n, V, P, E) of row j+LEAD.  Every offset is a multiple of 16 bytes (W * sizeof(T) >= 128).
template <typename T, int VEC, int MODEL, bool DRIVE>
struct StepSmem {
    using C = typename Cx<T>::type;
    static constexpr uint32_t NC = model_spinor(MODEL) ? 2 : 1;
    static constexpr bool RES = model_reservoir(MODEL);
    static constexpr uint32_t W = 32 * VEC;
    static constexpr uint32_t PSI = 0;
    static constexpr uint32_t N = PSI + NC * W * sizeof(C);
    static constexpr uint32_t V = N + (RES ? NC * W * sizeof(T) : 0);
    static constexpr uint32_t P = V + W * sizeof(T);
    static constexpr uint32_t E = P + (RES ? W * sizeof(T) : 0);
    static constexpr uint32_t STAGE = E + (DRIVE ? W * sizeof(C) : 0);
    static constexpr uint32_t DEPTH = step_ring_depth(sizeof(T) == 8, MODEL);
    static constexpr uint32_t BARS = PHX_STEP_WARPS * DEPTH * 8;          // mbarriers, at the start
    static constexpr uint32_t CTA = BARS + PHX_STEP_WARPS * DEPTH * STAGE;
};

// MINW: resident warps per SM the register budget is sized for.  ISO: dx == dy (scalar and reservoir models only).
// DRIVE: coherent drive E(r) exp(-i omega t) (reading Q17), shared by both components.
// BULK: rows are fetched by TMA bulk copies into a shared-memory ring instead of register loads (periodic boundaries only).
// XCH: the warps of a CTA (a.wpc of them, at most PHX_STEP_XWARPS) tile the WHOLE periodic row, nx = wpc * W, and exchange the
// one column a stage needs from the neighbouring strip through shared memory instead of recomputing 4 + 4 halo columns:
// every lane owns output columns (a 256-wide grid of cfg5 costs 4 strips of 64 columns instead of 5).  What a warp consumes in
// the iteration with front row j (the cells of psi[j], y2[j-1], y3[j-2], y4[j-3] next to its strip) its neighbours produced in
// iteration j-1 and left in slot (j-1) & 1 of a two-slot ring; a warp enters iteration j once both neighbours have finished
// j-1 (a progress counter per warp, polled in shared memory), so the warps of a row drift by less than one iteration and two
// slots suffice.  Scalar and reservoir models (the TE-TM corners would need a neighbour's row of the SAME iteration), periodic.
// UNITH: hbar = 1 exactly, so that 1/hbar times the potential is the potential (phx_deriv.cuh): one FP32 instruction fewer per
// cell and stage of the 17 the scalar model issues.
template <typename T, int VEC, int MODEL, bool NOISE, bool ZBC, bool ISO, bool DRIVE, int MINW, bool BULK, bool XCH = false,
          bool UNITH = false>
__global__ void __launch_bounds__(XCH ? 32 * PHX_STEP_XWARPS : 32 * PHX_STEP_WARPS, XCH ? 1 : MINW / PHX_STEP_WARPS)
step_kernel(const __grid_constant__ StepArgs<T> a) {
    using namespace stepk;
    using C = typename Cx<T>::type;
    constexpr bool SPINOR = model_spinor(MODEL);
    constexpr bool RES = model_reservoir(MODEL);
    constexpr int NC = SPINOR ? 2 : 1;
    constexpr int W = 32 * VEC, OUTW = XCH ? W : W - 8;
    constexpr int LEAD = XCH ? step_xch_lead(sizeof(T) == 8, MODEL, VEC) : PHX_STEP_LEAD, RING = 4 + LEAD;
    static_assert(!(BULK && ZBC), "the bulk-copy fetch path is built for periodic boundaries");
    static_assert(!(XCH && (ZBC || SPINOR)), "the exchanging strips are built for periodic scalar / reservoir grids");
    static_assert(!(XCH && BULK && !step_ring_cpasync(sizeof(T) == 8, MODEL, VEC)), "exchanging strips take the cp.async flavour of the ring only");
    const Geom& g = a.geo;
    const Coef<T>& k = a.k;
    const int nx = g.nx, ny = g.ny;

    // Programmatic dependent launch (a.pdl, set by the host for the second and later steps of a captured graph): the CTAs of
    // this grid may be scheduled while the previous step's grid is still running and wait here until it has completed and its
    // writes are visible -- the launch latency between two steps is hidden, nothing else changes (every global access of this
    // kernel, the step counter included, comes after the wait).  Both instructions do nothing in an ordinary launch.
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");
    const int lane = threadIdx.x & 31;
    const int strip = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const uint64_t step = *a.step_in;
    if (blockIdx.x == 0 && blockIdx.y == 0 && blockIdx.z == 0 && threadIdx.x == 0 && a.x0 == 0) *a.step_out = step + 1;
    if (!XCH && strip >= a.strips) return;   // warp-uniform
    // exchanging strips: the ring of edge cells [2 slots][4 arrays: psi, y2, y3, y4][warp][side: 0 = first cell, 1 = last cell of
    // the strip] and the progress counters (front row of the last iteration a warp has finished)
    typename Cx<T>::type* xe = nullptr;
    int* xp = nullptr;
    constexpr int XARR = PHX_STEP_XWARPS * 2;
    if constexpr (XCH) {
        __shared__ typename Cx<T>::type xedge_s[2 * 4 * XARR];
        __shared__ int xprog_s[PHX_STEP_XWARPS];
        xe = xedge_s;
        xp = xprog_s;
        if (threadIdx.x < PHX_STEP_XWARPS) xprog_s[threadIdx.x] = INT_MIN;
        __syncthreads();
    }

    // ---- columns of this lane ----------------------------------------------------------------------------------
    const int xl = a.x0 + strip * OUTW - (XCH ? 0 : 4) + lane * VEC;   // unwrapped column of the lane's first cell
    int xg = xl;                                     // column actually addressed
    bool inx = true;                                 // false: outside a zero boundary
    if (xl < 0 || xl >= nx) {
        if (ZBC && g.bc_x) { inx = false; xg = 0; }
        else { xg = xl % nx; if (xg < 0) xg += nx; }
    }
    const bool st_lane = XCH || (lane * VEC >= 4 && lane * VEC < W - 4 && xl < nx);   // lane owns output columns

    // ---- rows of this chunk ------------------------------------------------------------------------------------
    const int r0 = blockIdx.y * a.ly;
    const int r1 = min(r0 + a.ly, ny);
    const size_t boff = (size_t)blockIdx.z * g.plane;
    const bool zy = ZBC && g.bc_y;

    // drive: q_s = (1/hbar) exp(-i omega t_s) at the stage times t, t + dt/2, t + dt, t = step dt; the phase is evaluated
    // in double and rounded to T (reading Q17)
    C q1 = mk<T>(T(0), T(0)), q23 = q1, q4 = q1;
    if constexpr (DRIVE) {
        auto phase = [&](double cs) {
            double sn, cn;
            sincos(-k.omega * (((double)step + cs) * k.dt_d), &sn, &cn);
            return mk<T>(k.ih * (T)cn, k.ih * (T)sn);
        };
        q1 = phase(0.0); q23 = phase(0.5); q4 = phase(1.0);
    }

    // ---- base pointers of this realisation (warp-uniform); rows and columns are addressed by 32-bit cell offsets ----
    const C* pin[NC];
    C* pout[NC];
    const T* nin[NC];
    T* nout_p[NC];
#pragma unroll
    for (int s = 0; s < NC; ++s) {
        pin[s] = a.psi_in[s] + boff;
        pout[s] = a.psi_out[s] + boff;
        nin[s] = RES ? a.n_in[s] + boff : nullptr;
        nout_p[s] = RES ? a.n_out[s] + boff : nullptr;
    }
    const T* Vp = a.V;
    const T* Pp = RES ? a.P : nullptr;
    const C* Ep = DRIVE ? a.E : nullptr;
    // keep the bases as they are: one 64-bit register pair each, every access = base + (32-bit cell offset) * size
#pragma unroll
    for (int s = 0; s < NC; ++s) {
        asm volatile("" : "+l"(pin[s]), "+l"(pout[s]));
        if (RES) asm volatile("" : "+l"(nin[s]), "+l"(nout_p[s]));
    }
    asm volatile("" : "+l"(Vp), "+l"(Pp), "+l"(Ep));

    // ---- register rings (slot of row q = q mod RING; see the note above) ---------------------------------------------
    const C czero = mk<T>(T(0), T(0));
    C psr[NC][RING][VEC];                   // psi(t): rows j-2 .. j+1 live, row j+2 in flight
    C y2r[NC][RING][VEC];                   // stage-2 input: rows j-2, j-1 carried, row j produced
    C y3r[NC][RING][VEC];                   // stage-3 input: rows j-3, j-2 carried, row j-1 produced
    C y4r[NC][RING][VEC];                   // stage-4 input: rows j-4, j-3 carried, row j-2 produced
    C accr[NC][RING][VEC];                  // running sum of Eq. (6): row j produced, rows j-1 .. j-3 updated / consumed
    T Vr[RING][VEC], Pr[RING][VEC];         // V, P: rows j-3 .. j live, row j+1 in flight
    C Er[RING][VEC];                        // drive amplitude, as V
    T nr[NC][RING][VEC];                    // reservoir n(t): rows j-3 .. j live, row j+1 in flight
    T n2r[NC][RING][VEC], n3r[NC][RING][VEC], n4r[NC][RING][VEC];   // reservoir stage inputs (cell-local)
    T naccr[NC][RING][VEC];                 // reservoir running sum
#pragma unroll
    for (int r = 0; r < RING; ++r) {
#pragma unroll
        for (int i = 0; i < VEC; ++i) {
#pragma unroll
            for (int s = 0; s < NC; ++s) {
                psr[s][r][i] = czero; y2r[s][r][i] = czero; y3r[s][r][i] = czero; y4r[s][r][i] = czero; accr[s][r][i] = czero;
                nr[s][r][i] = T(0); n2r[s][r][i] = T(0); n3r[s][r][i] = T(0); n4r[s][r][i] = T(0); naccr[s][r][i] = T(0);
            }
            Vr[r][i] = T(0); Pr[r][i] = T(0); Er[r][i] = czero;
        }
    }

    // ---- row bookkeeping: the wrapped index of the row being fetched and the cell offsets (within one plane, < 2^31:
    // checked by the launch plan) of the lane's first cell in the rows fetched and stored, advanced by one row per iteration
    const uint32_t plane = (uint32_t)g.plane;
    const int j0 = r0 - 3;                  // first front row: stage 1 starts on row r0-3, stage 4 reaches row r0 three rows later
    int qw = j0 - 1;                        // row being fetched (wrapped unless outside a zero boundary)
    if (!zy) { qw %= ny; if (qw < 0) qw += ny; }
    uint32_t ew = (uint32_t)(qw * nx + xg); // its cell offset (modulo 2^32 while the row is outside a zero boundary)
    uint32_t ewp = 0;                       // cell offset of the row fetched before it
    bool okprev = !ZBC;
    uint32_t est = (uint32_t)((j0 - 3) * nx + xl);   // cell offset in the row stored in this iteration (row j-3), never wrapped
    // rows further ahead are pulled from DRAM into L2 by prefetch instructions, PF rows ahead of the register fetch
    constexpr int PF = PHX_STEP_PF_ROWS;
    const int pfr = ny >= PF ? PF : 0;      // (a grid shorter than the prefetch distance prefetches the row it is fetching)
    const uint32_t epf = (uint32_t)(pfr * nx);
    if (PF > 0 && inx) {
        // warm-up: the first PF rows of the chunk
        int q = qw;
        uint32_t e = ew;
        for (int r = 0; r < PF; ++r) {
            if (!zy || (q >= 0 && q < ny)) {
#pragma unroll
                for (int s = 0; s < NC; ++s) {
                    prefetch_l2(pin[s] + e);
                    if (RES) prefetch_l2(nin[s] + e);
                }
                if (Vp) prefetch_l2(Vp + e);
                if (Pp) prefetch_l2(Pp + e);
                if (DRIVE) prefetch_l2(Ep + e);
            }
            ++q; e += nx;
            if (!zy && q == ny) { q = 0; e -= plane; }
        }
    }

    // ---- pipeline fill: psi rows j0-1, j0, j0+1 and the row-local inputs (V, P, n) of row j0 ----------------------------------
#pragma unroll
    for (int d = -1; d <= LEAD; ++d) {
        constexpr int R2 = 2 * RING;
        const bool okq = !ZBC || (inx && (!zy || (qw >= 0 && qw < ny)));
#pragma unroll
        for (int s = 0; s < NC; ++s) {
            if (okq) ldc<VEC>(pin[s] + ew, psr[s][(d + R2) % RING]);
        }
        if (d >= 0 && d < LEAD && okq) {
            if (Vp) ldr<VEC>(Vp + ew, Vr[(d + R2) % RING]);
            if (Pp) ldr<VEC>(Pp + ew, Pr[(d + R2) % RING]);
            if (DRIVE) ldc<VEC>(Ep + ew, Er[(d + R2) % RING]);
            if constexpr (RES) {
#pragma unroll
                for (int s = 0; s < NC; ++s) ldr<VEC>(nin[s] + ew, nr[s][(d + R2) % RING]);
            }
        }
        ewp = ew;
        okprev = okq;
        ++qw; ew += nx;
        if (!zy && qw == ny) { qw = 0; ew -= plane; }
    }

    // ---- exchanging strips: neighbours, this lane's slots, and psi[j0] (the centre row of stage 1 in the first iteration)
    // published as the product of "iteration j0 - 1" ---------------------------------------------------------------------------
    int xleft = 0, xright = 0, xrd = 0, xwr = 0;
    const bool xlane = lane == 0 || lane == 31;
    if constexpr (XCH) {
        const int nw = blockDim.x >> 5;
        xleft = strip == 0 ? nw - 1 : strip - 1;
        xright = strip == nw - 1 ? 0 : strip + 1;
        xrd = lane == 0 ? xleft * 2 + 1 : xright * 2;   // lane 0 reads the last cell of the strip to the west, lane 31 the first of the strip to the east
        xwr = strip * 2 + (lane == 0 ? 0 : 1);
        if (xlane) xst(xe + (((j0 - 1) & 1) * 4 + 0) * XARR + xwr, lane == 0 ? psr[0][0][0] : psr[0][0][VEC - 1]);
#if PHX_XCH_SYNC == 1
        __syncthreads();
#else
        if (lane == 0) xst_flag(xp + strip, j0 - 1);
#endif
    }

    // ---- bulk-copy fetch path: the ring, its mbarriers and the issuer's state ------------------------------------------------
    using SM = StepSmem<T, VEC, MODEL, DRIVE>;
    constexpr int DEPTH = (int)SM::DEPTH;
    constexpr bool CPA = step_ring_cpasync(sizeof(T) == 8, MODEL, VEC);      // flavour of the ring: cp.async per lane, or TMA bulk copies
    extern __shared__ __align__(128) unsigned char step_smem[];
    uint32_t bar0 = 0, ring0 = 0;                       // shared-window addresses of this warp's mbarriers and stages
    const unsigned char* ringp = nullptr;
    int fi = 0, fc = 0, ntot = 0;                       // next fetch to issue / to consume; fetches in all (= row iterations)
    int qi = qw, qip = qw;                              // wrapped row of the psi / of the row-local inputs of fetch fi
    uint32_t txbytes = 0;
    int c0 = 0;                                         // wrapped first column of the strip
    if constexpr (BULK) {
        const int warp = threadIdx.x >> 5;
        bar0 = smem_u32(step_smem) + warp * DEPTH * 8;
        ringp = step_smem + SM::BARS + warp * DEPTH * SM::STAGE;
        ring0 = smem_u32(ringp);
        if constexpr (!CPA) {
            if (lane == 0) {
#pragma unroll
                for (int d = 0; d < DEPTH; ++d) mbar_init(bar0 + d * 8, 1);
                asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
            }
            __syncwarp();
        }
        ntot = ((r1 + 2 - j0) / RING + 1) * RING;
        qip = qw == 0 ? ny - 1 : qw - 1;
        c0 = (strip * OUTW - 4) % nx;
        if (c0 < 0) c0 += nx;
        txbytes = (uint32_t)W * (uint32_t)(NC * sizeof(C) + (RES ? NC * sizeof(T) : 0) + (Vp ? sizeof(T) : 0) + (Pp ? sizeof(T) : 0) +
                                           (DRIVE ? sizeof(C) : 0));
    }
    // issues fetch fi (psi row qi of every component, row-local inputs of row qip) into stage fi mod DEPTH; a strip that
    // crosses the periodic x edge is copied in two pieces (the launch plan takes this path only for nx >= W)
    const uint32_t lead = lane == 0;
    const int len1 = min((int)W, nx - c0), len2 = W - len1;
    auto issue_fetch = [&]() {
        if constexpr (CPA) {
            const uint32_t dst = ring0 + ((uint32_t)fi % DEPTH) * SM::STAGE;
            const uint32_t eq = (uint32_t)qi * (uint32_t)nx + (uint32_t)xg, ep = (uint32_t)qip * (uint32_t)nx + (uint32_t)xg;
#pragma unroll
            for (int s = 0; s < NC; ++s) {
                ring_cp<VEC * sizeof(C)>(dst + SM::PSI + s * W * sizeof(C), lane, pin[s] + eq);
                if constexpr (RES) cpasync<VEC * sizeof(T)>(dst + SM::N + (s * W + lane * VEC) * sizeof(T), nin[s] + ep);
            }
            if (Vp) cpasync<VEC * sizeof(T)>(dst + SM::V + lane * VEC * sizeof(T), Vp + ep);
            if (Pp) cpasync<VEC * sizeof(T)>(dst + SM::P + lane * VEC * sizeof(T), Pp + ep);
            if constexpr (DRIVE) ring_cp<VEC * sizeof(C)>(dst + SM::E, lane, Ep + ep);
            asm volatile("cp.async.commit_group;" ::: "memory");
            ++fi;
            qip = qi;
            if (++qi == ny) qi = 0;
            return;
        }
        const uint32_t slot = (uint32_t)fi % DEPTH, bar = bar0 + slot * 8, dst = ring0 + slot * SM::STAGE;
        mbar_expect_tx(bar, txbytes, lead);
        const uint32_t eq = (uint32_t)qi * (uint32_t)nx, ep = (uint32_t)qip * (uint32_t)nx;
#pragma unroll
        for (int s = 0; s < NC; ++s) {
            bulk_g2s(dst + SM::PSI + s * W * sizeof(C), pin[s] + eq + c0, len1 * sizeof(C), bar, lead);
            if constexpr (RES) bulk_g2s(dst + SM::N + s * W * sizeof(T), nin[s] + ep + c0, len1 * sizeof(T), bar, lead);
        }
        if (Vp) bulk_g2s(dst + SM::V, Vp + ep + c0, len1 * sizeof(T), bar, lead);
        if (Pp) bulk_g2s(dst + SM::P, Pp + ep + c0, len1 * sizeof(T), bar, lead);
        if constexpr (DRIVE) bulk_g2s(dst + SM::E, Ep + ep + c0, len1 * sizeof(C), bar, lead);
        if (len2 > 0) {
#pragma unroll
            for (int s = 0; s < NC; ++s) {
                bulk_g2s(dst + SM::PSI + (s * W + len1) * sizeof(C), pin[s] + eq, len2 * sizeof(C), bar, lead);
                if constexpr (RES) bulk_g2s(dst + SM::N + (s * W + len1) * sizeof(T), nin[s] + ep, len2 * sizeof(T), bar, lead);
            }
            if (Vp) bulk_g2s(dst + SM::V + len1 * sizeof(T), Vp + ep, len2 * sizeof(T), bar, lead);
            if (Pp) bulk_g2s(dst + SM::P + len1 * sizeof(T), Pp + ep, len2 * sizeof(T), bar, lead);
            if constexpr (DRIVE) bulk_g2s(dst + SM::E + len1 * sizeof(C), Ep + ep, len2 * sizeof(C), bar, lead);
        }
        ++fi;
        qip = qi;
        if (++qi == ny) qi = 0;
    };
    uint32_t ready = 0;                                 // has the stage of the next iteration landed? (tested one iteration early)
    if constexpr (BULK) {
        for (int d = 0; d < DEPTH - 1 && fi < ntot; ++d) issue_fetch();
    }

    // ---- row loop: one pass = RING front rows j0 + RING*k + ph.  Each phase is straight-line code (no branch around the
    // fetch or the four stages), so that the scheduler sees the loads and their consumers in one block. -------------------------
#define SL(d) ((ph + (d) + 2 * RING) % RING)     // ring slot of row j+d
#pragma unroll 1
    for (int jb = j0; jb <= r1 + 2; jb += RING) {
#pragma unroll
        for (int ph = 0; ph < RING; ++ph) {
            const int j = jb + ph;          // front row of this iteration
            if constexpr ((!BULK || (PHX_RING_EXIT && step_ring_cpasync(sizeof(T) == 8, MODEL, VEC))) && !XCH && step_early_exit(sizeof(T) == 8, MODEL, VEC)) {
                if (ph > 0 && j > r1 + 2) break;   // (warp-uniform) the chunk is done: row r1-1 was stored in the iteration with front row r1+2
            }
            C xin[4];                       // (XCH) the neighbours' cells next to this lane's strip: of psi[j], y2[j-1], y3[j-2], y4[j-3]
            if constexpr (XCH) {
#if PHX_XCH_SYNC == 0
                while (xld_flag(xp + xleft) < j - 1 || xld_flag(xp + xright) < j - 1) { }   // both finished iteration j-1
#endif
#pragma unroll
                for (int q = 0; q < 4; ++q) xin[q] = xld(xe + (((j - 1) & 1) * 4 + q) * XARR + xrd);
            }
            if (PF > 0 && !BULK) {
                if (!ZBC) {
                    uint32_t e = ew + epf;                   // row qw + pfr, wrapped
                    if (qw + pfr >= ny) e -= plane;
#pragma unroll
                    for (int s = 0; s < NC; ++s) {
                        prefetch_l2(pin[s] + e);
                        if (RES) prefetch_l2(nin[s] + e);
                    }
                    if (Vp) prefetch_l2(Vp + e);
                    if (Pp) prefetch_l2(Pp + e);
                    if (DRIVE) prefetch_l2(Ep + e);
#if PHX_STEP_PF1_ROWS > 0
                    // L2 -> L1: the row the register fetch takes PF1 iterations from now (its L2 latency is then off the fetch)
                    uint32_t e1 = ew + (uint32_t)(PHX_STEP_PF1_ROWS * nx);
                    if (qw + PHX_STEP_PF1_ROWS >= ny) e1 -= plane;
#pragma unroll
                    for (int s = 0; s < NC; ++s) {
                        prefetch_l1(pin[s] + e1);
                        if (RES) prefetch_l1(nin[s] + e1);
                    }
                    if (Vp) prefetch_l1(Vp + e1);
                    if (Pp) prefetch_l1(Pp + e1);
#endif
                } else if (inx && (j + 1 + LEAD + pfr <= r1 + 3) && qw + pfr < ny && qw + pfr >= 0) {
#pragma unroll
                    for (int s = 0; s < NC; ++s) {
                        prefetch_l2(pin[s] + ew + epf);
                        if (RES) prefetch_l2(nin[s] + ew + epf);
                    }
                    if (Vp) prefetch_l2(Vp + ew + epf);
                    if (Pp) prefetch_l2(Pp + ew + epf);
                    if (DRIVE) prefetch_l2(Ep + ew + epf);
                }
            }
            // ---- fetch: psi row j+2; row-local inputs (V, P, n) of row j+1 -------------------------------------------------
            // Periodic: every (wrapped) row is readable, so the fetch is unconditional (rows past r1+3 are fetched and not
            // used).  Zero boundaries: a row or column outside the grid reads as 0.
            const bool okq = !ZBC || (inx && (j + 1 + LEAD <= r1 + 3) && (!zy || (qw >= 0 && qw < ny)));
            if constexpr (BULK) {
                // the stage of this iteration has landed (phase parity of its mbarrier); registers <- shared memory
                const uint32_t slot = (uint32_t)fc % DEPTH;
                if constexpr (CPA) asm volatile("cp.async.wait_group %0;" ::"n"(DEPTH - 2) : "memory");   // the oldest group -- this iteration's row -- has landed
                else if (!ready) mbar_wait(bar0 + slot * 8, ((uint32_t)fc / DEPTH) & 1u);                 // (rare: the copies run DEPTH - 1 rows ahead)
                const unsigned char* st = ringp + slot * SM::STAGE;
#pragma unroll
                for (int s = 0; s < NC; ++s) {
                    if constexpr (CPA) ring_ld<VEC>(st + SM::PSI + s * W * sizeof(C), lane, psr[s][SL(1 + LEAD)]);
                    else ldsc<VEC>(reinterpret_cast<const C*>(st + SM::PSI) + s * W + lane * VEC, psr[s][SL(1 + LEAD)]);
                    if constexpr (RES) ldsr<VEC>(reinterpret_cast<const T*>(st + SM::N) + s * W + lane * VEC, nr[s][SL(LEAD)]);
                }
                if (Vp) ldsr<VEC>(reinterpret_cast<const T*>(st + SM::V) + lane * VEC, Vr[SL(LEAD)]);
                if (Pp) ldsr<VEC>(reinterpret_cast<const T*>(st + SM::P) + lane * VEC, Pr[SL(LEAD)]);
                if constexpr (DRIVE) {
                    if constexpr (CPA) ring_ld<VEC>(st + SM::E, lane, Er[SL(LEAD)]);
                    else ldsc<VEC>(reinterpret_cast<const C*>(st + SM::E) + lane * VEC, Er[SL(LEAD)]);
                }
                ++fc;
                if constexpr (!CPA) ready = mbar_test(bar0 + ((uint32_t)fc % DEPTH) * 8, ((uint32_t)fc / DEPTH) & 1u);
            } else {
#pragma unroll
            for (int s = 0; s < NC; ++s) {
                if (ZBC) {
#pragma unroll
                    for (int i = 0; i < VEC; ++i) psr[s][SL(1 + LEAD)][i] = czero;
                }
                if (okq) ldc<VEC>(pin[s] + ew, psr[s][SL(1 + LEAD)]);
            }
            if (ZBC) {              // (periodic without V or P: the slots keep the zeros they were initialised with)
#pragma unroll
                for (int i = 0; i < VEC; ++i) { Vr[SL(LEAD)][i] = T(0); Pr[SL(LEAD)][i] = T(0); Er[SL(LEAD)][i] = czero; }
            }
            if (okprev) {
                if (Vp) ldr<VEC>(Vp + ewp, Vr[SL(LEAD)]);
                if (Pp) ldr<VEC>(Pp + ewp, Pr[SL(LEAD)]);
                if (DRIVE) ldc<VEC>(Ep + ewp, Er[SL(LEAD)]);
            }
            if constexpr (RES) {
#pragma unroll
                for (int s = 0; s < NC; ++s) {
                    if (ZBC) {
#pragma unroll
                        for (int i = 0; i < VEC; ++i) nr[s][SL(LEAD)][i] = T(0);
                    }
                    if (okprev) ldr<VEC>(nin[s] + ewp, nr[s][SL(LEAD)]);
                }
            }
            }

            {
                // in-domain flags of the rows whose next stage input is written (zero boundaries: 0 outside the grid)
                const bool in1 = !ZBC || (inx && (!zy || (j >= 0 && j < ny)));
                const bool in2 = !ZBC || (inx && (!zy || (j - 1 >= 0 && j - 1 < ny)));
                const bool in3 = !ZBC || (inx && (!zy || (j - 2 >= 0 && j - 2 < ny)));
                Nbhd<T> nb[NC][VEC];
                Diff<T> df[NC][VEC];
                auto O = [](int s) { return SPINOR ? 1 - s : 0; };            // index of the other component
                auto diffs = [&k](const Nbhd<T> (&nb)[NC][VEC], Diff<T> (&df)[NC][VEC]) {
#pragma unroll
                    for (int s = 0; s < NC; ++s) {
#pragma unroll
                        for (int i = 0; i < VEC; ++i) differences<T, SPINOR, ISO>(k, nb[s][i], df[s][i]);
                    }
                };

                // ---- stage 1: K1 on row j from psi rows j-1, j, j+1 (Eq. (2)) ---------------------------------------------
#pragma unroll
                for (int s = 0; s < NC; ++s) gather<T, VEC, SPINOR, XCH>(psr[s][SL(-1)], psr[s][SL(0)], psr[s][SL(1)], nb[s], lane, xin[0]);
                diffs(nb, df);
#pragma unroll
                for (int s = 0; s < NC; ++s) {
#pragma unroll
                    for (int i = 0; i < VEC; ++i) {
                        T Kn;
                        const T nres = RES ? nr[s][SL(0)][i] : T(0);
                        const C K = deriv<T, SPINOR, RES, DRIVE, ISO, UNITH>(k, nb[s][i].c, df[s][i], nb[O(s)][i].c, df[O(s)][i], s == 0, nres, Vr[SL(0)][i], Pr[SL(0)][i], Er[SL(0)][i], q1, Kn);
                        const C p = psr[s][SL(0)][i];
                        y2r[s][SL(0)][i] = in1 ? fma2s(k.hdt, K, p) : czero;
                        accr[s][SL(0)][i] = fma2s(k.dt6, K, p);
                        if (RES) { n2r[s][SL(0)][i] = nres + k.hdt * Kn; naccr[s][SL(0)][i] = nres + k.dt6 * Kn; }
                    }
                }

                if constexpr (XCH) {        // publish the edge cells of psi[j+1] and y2[j] (centre rows of stages 1, 2 in iteration j+1)
                    if (xlane) {
                        xst(xe + ((j & 1) * 4 + 0) * XARR + xwr, lane == 0 ? psr[0][SL(1)][0] : psr[0][SL(1)][VEC - 1]);
                        xst(xe + ((j & 1) * 4 + 1) * XARR + xwr, lane == 0 ? y2r[0][SL(0)][0] : y2r[0][SL(0)][VEC - 1]);
                    }
                }

                // ---- stage 2: K2 on row j-1 from y2 rows j-2, j-1, j (Eq. (3)) --------------------------------------------
#pragma unroll
                for (int s = 0; s < NC; ++s) gather<T, VEC, SPINOR, XCH>(y2r[s][SL(-2)], y2r[s][SL(-1)], y2r[s][SL(0)], nb[s], lane, xin[1]);
                diffs(nb, df);
#pragma unroll
                for (int s = 0; s < NC; ++s) {
#pragma unroll
                    for (int i = 0; i < VEC; ++i) {
                        T Kn;
                        const T nres = RES ? n2r[s][SL(-1)][i] : T(0);
                        const C K = deriv<T, SPINOR, RES, DRIVE, ISO, UNITH>(k, nb[s][i].c, df[s][i], nb[O(s)][i].c, df[O(s)][i], s == 0, nres, Vr[SL(-1)][i], Pr[SL(-1)][i], Er[SL(-1)][i], q23, Kn);
                        const C p = psr[s][SL(-1)][i];
                        y3r[s][SL(-1)][i] = in2 ? fma2s(k.hdt, K, p) : czero;
                        accr[s][SL(-1)][i] = fma2s(k.dt3, K, accr[s][SL(-1)][i]);
                        if (RES) { n3r[s][SL(-1)][i] = nr[s][SL(-1)][i] + k.hdt * Kn; naccr[s][SL(-1)][i] += k.dt3 * Kn; }
                    }
                }

                if constexpr (XCH) {
                    if (xlane) xst(xe + ((j & 1) * 4 + 2) * XARR + xwr, lane == 0 ? y3r[0][SL(-1)][0] : y3r[0][SL(-1)][VEC - 1]);
                }

                // ---- stage 3: K3 on row j-2 from y3 rows j-3, j-2, j-1 (Eq. (4)) ------------------------------------------
#pragma unroll
                for (int s = 0; s < NC; ++s) gather<T, VEC, SPINOR, XCH>(y3r[s][SL(-3)], y3r[s][SL(-2)], y3r[s][SL(-1)], nb[s], lane, xin[2]);
                diffs(nb, df);
#pragma unroll
                for (int s = 0; s < NC; ++s) {
#pragma unroll
                    for (int i = 0; i < VEC; ++i) {
                        T Kn;
                        const T nres = RES ? n3r[s][SL(-2)][i] : T(0);
                        const C K = deriv<T, SPINOR, RES, DRIVE, ISO, UNITH>(k, nb[s][i].c, df[s][i], nb[O(s)][i].c, df[O(s)][i], s == 0, nres, Vr[SL(-2)][i], Pr[SL(-2)][i], Er[SL(-2)][i], q23, Kn);
                        const C p = psr[s][SL(-2)][i];
                        y4r[s][SL(-2)][i] = in3 ? fma2s(k.dt, K, p) : czero;
                        accr[s][SL(-2)][i] = fma2s(k.dt3, K, accr[s][SL(-2)][i]);
                        if (RES) { n4r[s][SL(-2)][i] = nr[s][SL(-2)][i] + k.dt * Kn; naccr[s][SL(-2)][i] += k.dt3 * Kn; }
                    }
                }

                if constexpr (XCH) {
                    if (xlane) xst(xe + ((j & 1) * 4 + 3) * XARR + xwr, lane == 0 ? y4r[0][SL(-2)][0] : y4r[0][SL(-2)][VEC - 1]);
#if PHX_XCH_SYNC == 1
                    asm volatile("bar.sync 1, %0;" ::"r"((int)blockDim.x));   // iteration j's cells are out: the warps of the row step together
#else
                    if (lane == 0) xst_flag(xp + strip, j);                             // iteration j's cells are out
#endif
                }

                // ---- stage 4: K4 on row j-3 from y4 rows j-4, j-3, j-2; psi(t+dt) of Eq. (6) (+ dW of Eq. (22)) ----------
#pragma unroll
                for (int s = 0; s < NC; ++s) gather<T, VEC, SPINOR, XCH>(y4r[s][SL(-4)], y4r[s][SL(-3)], y4r[s][SL(-2)], nb[s], lane, xin[3]);
                diffs(nb, df);
                const int jr = j - 3;
                const bool st_row = jr >= r0 && jr < r1;
                uint4 wd_prev[VEC];                                 // the Philox words of a cell: (x, y) for psi_+, (z, w) for psi_-
#pragma unroll
                for (int s = 0; s < NC; ++s) {
                    C out[VEC];
                    T nout[VEC];
#pragma unroll
                    for (int i = 0; i < VEC; ++i) {
                        T Kn;
                        const T nres = RES ? n4r[s][SL(-3)][i] : T(0);
                        const C K = deriv<T, SPINOR, RES, DRIVE, ISO, UNITH>(k, nb[s][i].c, df[s][i], nb[O(s)][i].c, df[O(s)][i], s == 0, nres, Vr[SL(-3)][i], Pr[SL(-3)][i], Er[SL(-3)][i], q4, Kn);
                        out[i] = fma2s(k.dt6, K, accr[s][SL(-3)][i]);
                        nout[i] = RES ? naccr[s][SL(-3)][i] + k.dt6 * Kn : T(0);
                    }
                    if (NOISE) {
                        // dW of Eq. (22), for every lane and row in straight-line code (no branch around it), so that the integer
                        // work of Philox interleaves with the floating-point work of the stages; rows and lanes that are not
                        // stored draw words nobody uses (the counter is the cell index, so nothing shifts)
#pragma unroll
                        for (int i = 0; i < VEC; ++i) {
                            const uint32_t cell = (uint32_t)jr * (uint32_t)nx + (uint32_t)(xl + i);
                            const uint4 wd = s == 0 ? noise_words(a.seed, blockIdx.z, step, cell) : wd_prev[i];
                            if (SPINOR && s == 0) wd_prev[i] = wd;
                            const T nt = RES ? nr[s][SL(-3)][i] : T(0);      // reservoir at the start of the step
                            const T var = k.sig2 * (T(2) * k.hgc + k.Rr * nt);
                            out[i] = add2(out[i], s == 0 ? noise_increment_sfu(wd.x, wd.y, var) : noise_increment_sfu(wd.z, wd.w, var));
                        }
                    }
                    if (st_row && st_lane) {
                        stc<VEC>(pout[s] + est, out);
                        if constexpr (RES) str<VEC>(nout_p[s] + est, nout);
                    }
                }
            }

            // ---- next row -----------------------------------------------------------------------------------------------
            if constexpr (BULK) {
                // the stage read in the previous iteration is free (its registers were consumed by this iteration's stages):
                // refill it with the row DEPTH - 1 iterations ahead
                if constexpr (CPA) {
                    issue_fetch();      // (always: one commit group per iteration keeps wait_group's count aligned)
                } else {
                    __syncwarp();
                    if (fi < ntot) issue_fetch();
                }
            }
            ewp = ew;
            okprev = okq;
            ++qw; ew += nx; est += nx;
            if (!zy && qw == ny) { qw = 0; ew -= plane; }
        }
    }
#undef SL
}

}  // namespace phx
