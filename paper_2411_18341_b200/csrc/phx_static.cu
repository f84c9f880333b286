// phx_static.cu -- phx_step_rk4_static: fixed-step RK4 (Eqs. (2)-(6)) of the scalar model Eq. (1)
// for callers that cannot allocate: no handle, no caller workspace, no cudaMalloc / cudaFree and no allocating
// library routine anywhere on the path (code under CUDA-graph capture, tight serving loops, harnesses that forbid allocation).
// The kernels are the fused per-stage kernels of variant STAGE (phx_stage.cuh), unchanged; what the
// handle keeps in the caller's workspace -- the two stage buffers y_a, y_b, the running sum of Eq. (6) and the step-counter
// slots -- lives instead in the file-scope device array below, of a fixed, modest size.  Every GPU that loads libphx.so
// holds those PHX_STATIC_SCRATCH_BYTES until the process exits.
//
// In host code the array's NAME is a host-side stand-in, not a device address: its device address is resolved once per
// device, with that device current, by cudaGetSymbolAddress in this file, and only that pointer is handed to the kernels.
// All calls share the array and it keeps the last call's contents: the counter slots are cleared by every call (the only
// part that must start from a known value -- every stage buffer is fully written before it is read), and two calls whose
// kernels overlap on the GPU (different streams) RACE on it.  Product code: shares nothing with oracle/.
#include "../../include/phx.h"

#include <cmath>
#include <cstring>
#include <mutex>

#include "phx_launch.h"
#include "phx_stage.cuh"

namespace {

static __device__ __align__(256) unsigned char phx_static_scratch[PHX_STATIC_SCRATCH_BYTES];

constexpr int MAX_DEVICES = 64;
std::mutex g_mutex;
unsigned char* g_scratch[MAX_DEVICES];      // device address of phx_static_scratch on device d (nullptr = not resolved yet)

// Device address of the scratch array on the CURRENT device (resolved once per device).
cudaError_t scratch_address(unsigned char** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_mutex);
    if (!g_scratch[dev]) {
        void* ptr = nullptr;
        e = cudaGetSymbolAddress(&ptr, phx_static_scratch);
        if (e != cudaSuccess) return e;
        if (!ptr) return cudaErrorInvalidSymbol;
        g_scratch[dev] = static_cast<unsigned char*>(ptr);
    }
    *out = g_scratch[dev];
    return cudaSuccess;
}

inline size_t align256(size_t v) { return (v + 255) / 256 * 256; }

// Canonical coefficients of DESIGN.md section 2, step 0 (the expressions of phx_set_params, each rounded once to T).
template <typename T>
bool fill_coef(const phx_params* p, double dx, double dy, phx::Coef<T>& k) {
    std::memset(&k, 0, sizeof(k));
    const double c[] = {p->hbar / (2.0 * p->m * dx * dx), p->hbar / (2.0 * p->m * dy * dy), 1.0 / p->hbar, p->g, p->gamma_c / 2.0,
                        p->dt, p->dt / 6.0, p->dt / 3.0, p->density_offset};
    for (double v : c)
        if (!std::isfinite(v)) return false;
    k.cx = (T)c[0]; k.cy = (T)c[1]; k.ih = (T)c[2]; k.g = (T)c[3]; k.hgc = (T)c[4];
    k.dt = (T)c[5];
    const double dt_t = (double)k.dt;           // (dt as the working type holds it, as the handle path stores it)
    k.hdt = (T)(0.5 * dt_t);
    k.dt6 = (T)c[6]; k.dt3 = (T)c[7]; k.doff = (T)c[8];
    const double r13 = (double)k.dt6 / (0.5 * dt_t);
    k.r13 = (T)r13;
    k.r13lo = (T)(r13 - (double)k.r13);
    k.omega = 0.0;
    k.dt_d = dt_t;
    return true;
}

template <typename T>
phx_status run(int nx, int ny, double dx, double dy, int bc_x, int bc_y, const phx_params* p, const void* V, const void* psi_in,
               void* psi_out, int64_t n_steps, cudaStream_t st) {
    using C = typename phx::Cx<T>::type;
    const size_t cells = (size_t)nx * (size_t)ny, plane_bytes = align256(cells * sizeof(C));
    if (3 * plane_bytes + 256 > (size_t)PHX_STATIC_SCRATCH_BYTES) return PHX_ERR_WORKSPACE;   // grid beyond the static scratch
    unsigned char* base = nullptr;
    if (scratch_address(&base) != cudaSuccess) { cudaGetLastError(); return PHX_ERR_CUDA; }

    phx::StageArgs<T> a;
    std::memset(&a, 0, sizeof(a));
    a.geo.nx = nx; a.geo.ny = ny; a.geo.batch = 1;
    a.geo.bc_x = bc_x; a.geo.bc_y = bc_y;
    a.geo.rows = 16;
    a.geo.plane = cells;
    if (!fill_coef<T>(p, dx, dy, a.k)) return PHX_ERR_INVALID_ARG;
    a.f.psi[0] = static_cast<C*>(psi_out);                       // the state is stepped in place in the caller's output array
    a.f.ya[0] = reinterpret_cast<C*>(base);
    a.f.yb[0] = reinterpret_cast<C*>(base + plane_bytes);
    a.f.acc[0] = reinterpret_cast<C*>(base + 2 * plane_bytes);
    a.f.step = reinterpret_cast<uint64_t*>(base + 3 * plane_bytes);
    a.f.V = static_cast<const T*>(V);
    a.seed = p->seed;

    if (psi_in != psi_out && cudaMemcpyAsync(psi_out, psi_in, cells * sizeof(C), cudaMemcpyDeviceToDevice, st) != cudaSuccess) {
        cudaGetLastError();
        return PHX_ERR_CUDA;
    }
    // the array keeps the last call's contents: the counter slots start every call at 0
    if (cudaMemsetAsync(a.f.step, 0, 256, st) != cudaSuccess) { cudaGetLastError(); return PHX_ERR_CUDA; }

    // launch geometry of variant STAGE (phx_api.cu: enqueue_step_stage)
    const int vec = (sizeof(T) == 4 && nx % 2 == 0) ? 2 : 1;
    const int tx = (nx + vec - 1) / vec;
    int bx = ((tx + 31) / 32) * 32;
    if (bx > 128) bx = 128;
    const int by = 128 / bx;
    const dim3 block(bx, by, 1);
    const dim3 grid((tx + bx - 1) / bx, (ny + a.geo.rows * by - 1) / (a.geo.rows * by), 1);
    for (int64_t s = 0; s < n_steps; ++s) {
        for (int stage = 1; stage <= 4; ++stage) {
            cudaError_t e;
            if constexpr (sizeof(T) == 4) e = phx::launch_stage_32_0(a, stage, false, vec, grid, block, st);
            else e = phx::launch_stage_64_0(a, stage, false, vec, grid, block, st);
            if (e != cudaSuccess) { cudaGetLastError(); return PHX_ERR_CUDA; }
        }
    }
    return PHX_OK;
}

}  // namespace

extern "C" phx_status phx_step_rk4_static(int32_t nx, int32_t ny, double dx, double dy, int32_t prec, int32_t bc_x, int32_t bc_y,
                                          const phx_params* p, const void* V, const void* psi_in, void* psi_out, int64_t n_steps,
                                          void* stream) {
    if (!p || !psi_in || !psi_out || nx < 3 || ny < 3 || n_steps < 0 || !(dx > 0) || !(dy > 0)) return PHX_ERR_INVALID_ARG;
    if (prec != PHX_C32 && prec != PHX_C64) return PHX_ERR_INVALID_ARG;
    if ((bc_x != 0 && bc_x != 1) || (bc_y != 0 && bc_y != 1)) return PHX_ERR_INVALID_ARG;
    if (!(p->dt > 0) || p->hbar == 0 || p->m == 0 || !std::isfinite(p->hbar) || !std::isfinite(p->m) || !std::isfinite(p->dt))
        return PHX_ERR_INVALID_ARG;
    if ((size_t)nx * (size_t)ny > (size_t)PHX_STATIC_SCRATCH_BYTES) return PHX_ERR_WORKSPACE;      // (before any size arithmetic)
    const cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (prec == PHX_C64) return run<double>(nx, ny, dx, dy, bc_x, bc_y, p, V, psi_in, psi_out, n_steps, st);
    return run<float>(nx, ny, dx, dy, bc_x, bc_y, p, V, psi_in, psi_out, n_steps, st);
}
