// phx_adaptive.cu -- adaptive Dormand-Prince 5(4) time stepping.  The paper names the method only
// ("higher-order methods like the RK-Fehlberg or Dormand-Prince can be used for systems requiring adaptive
// time-stepping", :488); tableau, error norm and controller are DESIGN.md reading Q20.
//
// One ATTEMPT = seven fused stage kernels and a one-thread controller kernel, all of them nodes of the body of a CUDA-graph
// WHILE node: the controller decides accept / reject, the next step size and whether the loop goes on
// (cudaGraphSetConditional) ON THE DEVICE -- the host enqueues one graph launch per phx_step_adaptive call and never reads
// anything back.
//   stage s (1..6): K_s = f(Y_s, t + c_s h) from the stage input with a one-cell halo (the derivative of phx_deriv.cuh, the
//                   same one the fused RK4 step uses); K_s is stored and, in the same pass, the next stage input
//                   Y_{s+1} = u + h sum_{j<=s} a_{s+1,j} K_j is formed (K_1..K_{s-1} re-read).  Y_7 is the candidate u_new.
//                   Stage 1 skips the derivative when K_1 is the K_7 of the last accepted step (FSAL).
//   stage 7:        K_7 = f(u_new, t + h); the error estimate E = h sum_j e_j K_j and the norm
//                   err = max |E| / (atol + rtol max(|u|, |u_new|)) over every cell / component / reservoir / realisation:
//                   block maximum, then one atomicMax on the bit pattern (non-negative doubles order like integers), so the
//                   result does not depend on the order of the reduction.
//   control:        accept iff err <= 1 (or the proposal is already h_min); q = floor(16 clamp(0.9 err^-1/5, 1/4, 4));
//                   h <- clamp(h_used q / 16); on accept t advances, u <-> u_new and K_1 <-> K_7 swap roles (a flag, no copy).
// Product code: shares nothing with oracle/.
#include "phx_adaptive.h"

#include <cuda_device_runtime_api.h>

#include "phx_deriv.cuh"

namespace phx {

namespace {

template <typename T>
__device__ __forceinline__ typename Cx<T>::type ldg_bc(const typename Cx<T>::type* p, int i, int j, const Geom& g) {
    // value at (i, j) under the boundary rule of PAPER.md:369: periodic (wrapped index) or zero (0 outside the grid)
    if (i < 0 || i >= g.nx) {
        if (g.bc_x) return mk<T>(T(0), T(0));
        i = i < 0 ? i + g.nx : i - g.nx;
    }
    if (j < 0 || j >= g.ny) {
        if (g.bc_y) return mk<T>(T(0), T(0));
        j = j < 0 ? j + g.ny : j - g.ny;
    }
    return p[(size_t)j * g.nx + i];
}

template <typename T> __device__ __forceinline__ T cabs_t(typename Cx<T>::type z) { return sqrt(z.x * z.x + z.y * z.y); }

// One stage (S = 1..7) of one attempt.  One thread per cell; block 32 x 8; blockIdx.z = realisation.
template <typename T, int MODEL, int S>
__global__ void __launch_bounds__(256) dp_stage_kernel(const __grid_constant__ DpArgs<T> a) {
    using C = typename Cx<T>::type;
    constexpr bool SPINOR = model_spinor(MODEL);
    constexpr bool RES = model_reservoir(MODEL);
    constexpr int NC = SPINOR ? 2 : 1;
    const Geom& g = a.geo;
    const Coef<T>& k = a.k;
    DpCtl* ctl = a.ctl;
    if (ctl->done) return;
    const int cur = ctl->cur;
    const bool k1_valid = ctl->k1_valid != 0;
    const T h = (T)ctl->hu;
    const double t_stage = ctl->t + (double)a.c[S - 1] * ctl->hu;

    const int i = blockIdx.x * 32 + threadIdx.x, j = blockIdx.y * 8 + threadIdx.y;
    const bool active = i < g.nx && j < g.ny;
    const size_t boff = (size_t)blockIdx.z * g.plane;
    const size_t cell = boff + (size_t)(active ? j : 0) * g.nx + (active ? i : 0);
    T ratio = T(0);

    if (active) {
        // wiring of this stage: where the stage input, the state u, the candidate u_new and K_1 / K_7 live
        const C* yin[NC]; C* yout[NC]; const C* u[NC]; const T* nin[NC]; T* nout[NC]; const T* un_[NC];
        C* K[7][NC]; T* Kn[7][NC];
#pragma unroll
        for (int s = 0; s < NC; ++s) {
            const C* us = a.S[cur][s];
            C* unew = a.S[1 - cur][s];
            u[s] = us;
            yin[s] = S == 1 ? us : (S == 7 ? unew : (S % 2 == 0 ? a.Y[0][s] : a.Y[1][s]));     // Y2, Y4, Y6 in Y[0]; Y3, Y5 in Y[1]
            yout[s] = S == 6 ? unew : (S % 2 == 1 ? a.Y[0][s] : a.Y[1][s]);
#pragma unroll
            for (int q = 0; q < 7; ++q) K[q][s] = q == 0 ? a.K[cur ? 6 : 0][s] : (q == 6 ? a.K[cur ? 0 : 6][s] : a.K[q][s]);
            if constexpr (RES) {
                const T* ns = a.Sn[cur][s];
                T* nnew = a.Sn[1 - cur][s];
                un_[s] = ns;
                nin[s] = S == 1 ? ns : (S == 7 ? nnew : (S % 2 == 0 ? a.Yn[0][s] : a.Yn[1][s]));
                nout[s] = S == 6 ? nnew : (S % 2 == 1 ? a.Yn[0][s] : a.Yn[1][s]);
#pragma unroll
                for (int q = 0; q < 7; ++q) Kn[q][s] = q == 0 ? a.Kn[cur ? 6 : 0][s] : (q == 6 ? a.Kn[cur ? 0 : 6][s] : a.Kn[q][s]);
            }
        }

        // ---- K_S = f(Y_S, t + c_S h) ----------------------------------------------------------------------------------
        C Ks[NC];
        T Kns[NC];
        const bool need_f = !(S == 1 && k1_valid);
        if (need_f) {
            Nbhd<T> nb[NC];
            Diff<T> df[NC];
#pragma unroll
            for (int s = 0; s < NC; ++s) {
                const C* p = yin[s] + boff;
                nb[s].c = p[(size_t)j * g.nx + i];
                nb[s].w = ldg_bc<T>(p, i - 1, j, g);
                nb[s].e = ldg_bc<T>(p, i + 1, j, g);
                nb[s].s = ldg_bc<T>(p, i, j - 1, g);
                nb[s].n = ldg_bc<T>(p, i, j + 1, g);
                if (SPINOR) {
                    const C ne = ldg_bc<T>(p, i + 1, j + 1, g), se = ldg_bc<T>(p, i + 1, j - 1, g);
                    const C nw = ldg_bc<T>(p, i - 1, j + 1, g), sw = ldg_bc<T>(p, i - 1, j - 1, g);
                    nb[s].D = sub2(sub2(ne, se), sub2(nw, sw));
                }
                differences<T, SPINOR, false>(k, nb[s], df[s]);
            }
            C q = mk<T>(T(0), T(0));
            C Ed = q;
            if (a.E) {
                double sn, cn;
                sincos(-k.omega * t_stage, &sn, &cn);
                q = mk<T>(k.ih * (T)cn, k.ih * (T)sn);
                Ed = a.E[(size_t)j * g.nx + i];
            }
            const T Vc = a.V ? a.V[(size_t)j * g.nx + i] : T(0);
            const T Pc = (RES && a.P) ? a.P[(size_t)j * g.nx + i] : T(0);
#pragma unroll
            for (int s = 0; s < NC; ++s) {
                const int o = SPINOR ? 1 - s : 0;
                const T nres = RES ? nin[s][cell] : T(0);
                Ks[s] = deriv<T, SPINOR, RES, true>(k, nb[s].c, df[s], nb[o].c, df[o], s == 0, nres, Vc, Pc, Ed, q, Kns[s]);
                K[S - 1][s][cell] = Ks[s];
                if (RES) Kn[S - 1][s][cell] = Kns[s];
            }
        } else {
#pragma unroll
            for (int s = 0; s < NC; ++s) {
                Ks[s] = K[0][s][cell];
                if (RES) Kns[s] = Kn[0][s][cell];
            }
        }

        if constexpr (S < 7) {
            // ---- Y_{S+1} = u + h sum_{j <= S} a_{S+1,j} K_j (row S of the tableau, 0-based) ---------------------------------
#pragma unroll
            for (int s = 0; s < NC; ++s) {
                C acc = mk<T>(T(0), T(0));
#pragma unroll
                for (int q = 0; q < S; ++q) acc = fma2s(a.a[S][q], q == S - 1 ? Ks[s] : K[q][s][cell], acc);
                yout[s][cell] = fma2s(h, acc, u[s][cell]);
                if constexpr (RES) {
                    T an = T(0);
#pragma unroll
                    for (int q = 0; q < S; ++q) an = fma(a.a[S][q], q == S - 1 ? Kns[s] : Kn[q][s][cell], an);
                    nout[s][cell] = fma(h, an, un_[s][cell]);
                }
            }
        } else {
            // ---- error estimate E = h sum_j e_j K_j and its ratio to the tolerance ------------------------------------------
#pragma unroll
            for (int s = 0; s < NC; ++s) {
                C E = mk<T>(T(0), T(0));
#pragma unroll
                for (int q = 0; q < 7; ++q) E = fma2s(a.e[q], q == 6 ? Ks[s] : K[q][s][cell], E);
                const T sc = (T)ctl->atol + (T)ctl->rtol * max(cabs_t<T>(u[s][cell]), cabs_t<T>(yin[s][cell]));
                ratio = max(ratio, abs(h) * cabs_t<T>(E) / sc);
                if constexpr (RES) {
                    T En = T(0);
#pragma unroll
                    for (int q = 0; q < 7; ++q) En = fma(a.e[q], q == 6 ? Kns[s] : Kn[q][s][cell], En);
                    const T scn = (T)ctl->atol + (T)ctl->rtol * max(abs(un_[s][cell]), abs(nin[s][cell]));
                    ratio = max(ratio, abs(h * En) / scn);
                }
            }
        }
    }

    if constexpr (S == 7) {
        // block maximum, then one atomicMax on the bit pattern of the (non-negative) double
        __shared__ double red[8];
        double r = (double)ratio;
        if (!(r == r)) r = 1.0e300;                                  // a NaN anywhere rejects the step
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) r = fmax(r, __shfl_xor_sync(0xffffffffu, r, o));
        if (threadIdx.x == 0) red[threadIdx.y] = r;
        __syncthreads();
        if (threadIdx.x == 0 && threadIdx.y == 0) {
            double m = red[0];
#pragma unroll
            for (int w = 1; w < 8; ++w) m = fmax(m, red[w]);
            atomicMax(&ctl->err_bits, (unsigned long long)__double_as_longlong(m));
        }
    }
}

// Sets up the first attempt of a call: the step to try, clipped so that the call lands on t_end, rounded once to T.
__device__ void dp_plan_attempt(DpCtl* c, bool prec32) {
    c->clipped = c->t + c->h >= c->t_end ? 1 : 0;
    const double hu = c->clipped ? c->t_end - c->t : c->h;
    c->hu = prec32 ? (double)(float)hu : hu;
    c->err_bits = 0ull;
}

__global__ void dp_setup_kernel(DpCtl* c, cudaGraphConditionalHandle handle, int prec32) {
    c->attempts = 0;
    c->log_count = 0;
    if (!(c->h > 0.0)) c->h = c->h_init;
    c->h = fmin(c->h_max, fmax(c->h_min, c->h));
    c->done = (c->t < c->t_end && c->max_attempts > 0) ? 0 : 1;
    dp_plan_attempt(c, prec32 != 0);
    cudaGraphSetConditional(handle, c->done ? 0u : 1u);
}

__global__ void dp_control_kernel(DpCtl* c, cudaGraphConditionalHandle handle, int prec32, int log_cap) {
    const double err = __longlong_as_double((long long)c->err_bits);
    const bool accept = err <= 1.0 || c->h <= c->h_min;
    double fac = err > 0.0 ? 0.9 * pow(err, -0.2) : 4.0;
    fac = fmin(4.0, fmax(0.25, fac));
    const int q = (int)floor(16.0 * fac);
    if (c->log_count < log_cap) {
        const long long n = c->log_count;
        c->log_accept[n] = accept ? 1 : 0;
        c->log_q[n] = q;
        c->log_h[n] = c->hu;
        c->log_err[n] = err;
    }
    c->log_count += 1;
    c->attempts += 1;
    c->err_last = err;
    if (accept) {
        c->t = c->clipped ? c->t_end : c->t + c->hu;
        c->cur ^= 1;                                               // u <-> u_new, K_1 <-> K_7 (FSAL)
        c->k1_valid = 1;
        c->n_accept += 1;
        if (!c->clipped) c->h = fmin(c->h_max, fmax(c->h_min, c->hu * (double)q / 16.0));
    } else {
        c->n_reject += 1;
        c->h = fmin(c->h_max, fmax(c->h_min, c->hu * (double)q / 16.0));
    }
    c->done = (c->t < c->t_end && c->attempts < c->max_attempts) ? 0 : 1;
    dp_plan_attempt(c, prec32 != 0);
    cudaGraphSetConditional(handle, c->done ? 0u : 1u);
}

// After the loop: the state goes back to the buffers the rest of the library reads (psi / n); K_1 is recomputed by the next call.
template <typename T>
__global__ void dp_finalize_kernel(const __grid_constant__ DpArgs<T> a, int nc, int res) {
    DpCtl* c = a.ctl;
    const int cur = c->cur;
    if (cur != 0) {
        const size_t n = a.geo.plane * (size_t)a.geo.batch;
        for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (size_t)gridDim.x * blockDim.x) {
            for (int s = 0; s < nc; ++s) {
                a.S[0][s][k] = a.S[1][s][k];
                if (res) a.Sn[0][s][k] = a.Sn[1][s][k];
            }
        }
    }
}

__global__ void dp_finalize_flags_kernel(DpCtl* c) {
    c->cur = 0;
    c->k1_valid = 0;
}

template <typename T, int MODEL>
cudaError_t launch_attempt_model(const DpArgs<T>& a, cudaStream_t st) {
    const dim3 block(32, 8, 1);
    const dim3 grid((a.geo.nx + 31) / 32, (a.geo.ny + 7) / 8, a.geo.batch);
    if (grid.y > 65535u) return cudaErrorInvalidConfiguration;
    dp_stage_kernel<T, MODEL, 1><<<grid, block, 0, st>>>(a);
    dp_stage_kernel<T, MODEL, 2><<<grid, block, 0, st>>>(a);
    dp_stage_kernel<T, MODEL, 3><<<grid, block, 0, st>>>(a);
    dp_stage_kernel<T, MODEL, 4><<<grid, block, 0, st>>>(a);
    dp_stage_kernel<T, MODEL, 5><<<grid, block, 0, st>>>(a);
    dp_stage_kernel<T, MODEL, 6><<<grid, block, 0, st>>>(a);
    dp_stage_kernel<T, MODEL, 7><<<grid, block, 0, st>>>(a);
    return cudaGetLastError();
}

}  // namespace

template <typename T>
cudaError_t dp_launch_attempt(const DpArgs<T>& a, int model, cudaStream_t st) {
    switch (model) {
        case M_SCALAR: return launch_attempt_model<T, M_SCALAR>(a, st);
        case M_RESERVOIR: return launch_attempt_model<T, M_RESERVOIR>(a, st);
        case M_SPINOR: return launch_attempt_model<T, M_SPINOR>(a, st);
        default: return launch_attempt_model<T, M_SPINOR_RESERVOIR>(a, st);
    }
}
template cudaError_t dp_launch_attempt<float>(const DpArgs<float>&, int, cudaStream_t);
template cudaError_t dp_launch_attempt<double>(const DpArgs<double>&, int, cudaStream_t);

cudaError_t dp_launch_setup(DpCtl* c, unsigned long long handle, int prec32, cudaStream_t st) {
    dp_setup_kernel<<<1, 1, 0, st>>>(c, (cudaGraphConditionalHandle)handle, prec32);
    return cudaGetLastError();
}

cudaError_t dp_launch_control(DpCtl* c, unsigned long long handle, int prec32, int log_cap, cudaStream_t st) {
    dp_control_kernel<<<1, 1, 0, st>>>(c, (cudaGraphConditionalHandle)handle, prec32, log_cap);
    return cudaGetLastError();
}

template <typename T>
cudaError_t dp_launch_finalize(const DpArgs<T>& a, int model, int n_sm, cudaStream_t st) {
    dp_finalize_kernel<T><<<4 * n_sm, 256, 0, st>>>(a, model_spinor(model) ? 2 : 1, model_reservoir(model) ? 1 : 0);
    dp_finalize_flags_kernel<<<1, 1, 0, st>>>(a.ctl);
    return cudaGetLastError();
}
template cudaError_t dp_launch_finalize<float>(const DpArgs<float>&, int, int, cudaStream_t);
template cudaError_t dp_launch_finalize<double>(const DpArgs<double>&, int, int, cudaStream_t);

}  // namespace phx
