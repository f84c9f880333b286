// phx_resident.cu -- variant RESIDENT: a small grid stays on chip for many RK4 steps of one launch
// (SURVEY.md section 8(a) "V-small persistent"; the paper's small-grid regime is bound by kernel-launch latency,
// PAPER.md:289, which CUDA graphs only soften, :195).
//
// One CTA of 512 threads owns one realisation (blockIdx.x).  A thread owns CPT cells (cell c = tid + k*512) and keeps
// their psi(t), the running sum of Eq. (6) and the reservoir values in registers for the whole launch.  The stage
// input y_s, of which a cell needs its four neighbours (Eq. (8)), lives in two shared-memory buffers that alternate:
// stage s reads buffer A and writes y_{s+1} into buffer B, one __syncthreads per stage, four per step (Eqs. (2)-(6),
// PAPER.md:53-62).  V, P and the four neighbour indices of every cell (periodic wrap, or a zero cell beyond a zero
// boundary) are staged in shared memory once.  HBM traffic: the state in at the first step and out at the
// last.  Scalar and reservoir models, both precisions, optional noise (Eq. (22)); no drive.
// The derivative is the one of variant STEP (phx_deriv.cuh).  Product code: shares nothing with oracle/.
//
// CLUSTER form (resident_cluster_kernel): one realisation spread over a thread-block cluster of 2-16 CTAs, each owning a slab
// of ny / cluster rows plus one halo row above and below in its own shared memory.  After a stage every CTA stores the first
// and last row it produced straight into its neighbours' halo rows through distributed shared memory
// (cluster.map_shared_rank), then the cluster barrier (barrier.cluster, ~380 cycles) takes the place of __syncthreads.  For a
// SINGLE small grid, which one SM steps too slowly (fp64: 64 lanes) and the fused step cannot step faster than a kernel
// launch per step allows (cfg1: 3.6 us per step).
#include "phx_common.cuh"
#include "phx_deriv.cuh"
#include "phx_philox.cuh"
#include "phx_launch.h"

#include <cooperative_groups.h>
#include <type_traits>

namespace phx {

constexpr int RES_NT = PHX_RESIDENT_THREADS;
// Scalar grids on a cluster: two stages per cluster barrier (resident_pair_kernel) instead of one.
#ifndef PHX_RESIDENT_PAIR
#define PHX_RESIDENT_PAIR 1
#endif
#ifndef PHX_RESIDENT_MAX_CLUSTER
#define PHX_RESIDENT_MAX_CLUSTER 16     // (beyond 8: the non-portable cluster size attribute, set at launch)
#endif

template <typename T, bool RES, bool NOISE, int CPT>
__global__ void __launch_bounds__(RES_NT, 1)
resident_kernel(const __grid_constant__ ResidentArgs<T> a) {
    using C = typename Cx<T>::type;
    extern __shared__ __align__(16) unsigned char smem[];
    const Geom& g = a.geo;
    const Coef<T>& k = a.k;
    const int nx = g.nx, ny = g.ny, N = nx * ny;
    // shared memory: two stage buffers of N + 1 complex (cell N holds 0), neighbour indices, V, P
    C* buf0 = reinterpret_cast<C*>(smem);
    C* buf1 = buf0 + (N + 1);
    ushort4* nbr = reinterpret_cast<ushort4*>(buf1 + (N + 1));      // w, e, s (row j-1), n (row j+1)
    T* Vs = reinterpret_cast<T*>(nbr + N);
    T* Ps = Vs + N;

    const int tid = threadIdx.x;
    const size_t boff = (size_t)blockIdx.x * g.plane;
    C* psi_g = a.psi + boff;
    T* n_g = RES ? a.n + boff : nullptr;
    const C czero = mk<T>(T(0), T(0));

    C psi[CPT], acc[CPT];
    T nn[CPT], nacc[CPT], nst[CPT];
#pragma unroll
    for (int q = 0; q < CPT; ++q) {
        const int c = tid + q * RES_NT;
        psi[q] = czero; acc[q] = czero; nn[q] = T(0); nacc[q] = T(0); nst[q] = T(0);
        if (c < N) {
            const int j = c / nx, i = c - j * nx;
            ushort4 nb;
            nb.x = (unsigned short)(i > 0 ? c - 1 : (g.bc_x ? N : c + nx - 1));
            nb.y = (unsigned short)(i < nx - 1 ? c + 1 : (g.bc_x ? N : c - nx + 1));
            nb.z = (unsigned short)(j > 0 ? c - nx : (g.bc_y ? N : c + N - nx));
            nb.w = (unsigned short)(j < ny - 1 ? c + nx : (g.bc_y ? N : c - N + nx));
            nbr[c] = nb;
            Vs[c] = a.V ? a.V[c] : T(0);
            Ps[c] = (RES && a.P) ? a.P[c] : T(0);
            psi[q] = psi_g[c];
            if (RES) nn[q] = n_g[c];
            buf0[c] = psi[q];
        }
    }
    if (tid == 0) { buf0[N] = czero; buf1[N] = czero; }
    __syncthreads();

    // one stage: K_s from the stage input in `in`; a_dt = a_s dt of Eqs. (3)-(5), w_dt = weight of K_s in Eq. (6)
    auto stage = [&](const C* in, C* out, auto stage_no, const uint64_t step) {
        constexpr int s = decltype(stage_no)::value;
        const T a_dt = s == 3 ? k.dt : k.hdt;
        const T w_dt = (s == 1 || s == 4) ? k.dt6 : k.dt3;
#pragma unroll
        for (int q = 0; q < CPT; ++q) {
            const int c = tid + q * RES_NT;
            if (c < N) {
                const ushort4 nb = nbr[c];
                Nbhd<T> h;
                h.c = s == 1 ? psi[q] : in[c];
                h.w = in[nb.x]; h.e = in[nb.y]; h.s = in[nb.z]; h.n = in[nb.w];
                Diff<T> df;
                differences<T, false, false>(k, h, df);
                const T nres = RES ? (s == 1 ? nn[q] : nst[q]) : T(0);
                T Kn;
                const C K = deriv<T, false, RES, false>(k, h.c, df, czero, df, true, nres, Vs[c], Ps[c], czero, czero, Kn);
                if (s == 1) {
                    acc[q] = fma2s(w_dt, K, psi[q]);
                    if (RES) nacc[q] = nn[q] + w_dt * Kn;
                } else if (s < 4) {
                    acc[q] = fma2s(w_dt, K, acc[q]);
                    if (RES) nacc[q] += w_dt * Kn;
                }
                if (s < 4) {
                    out[c] = fma2s(a_dt, K, psi[q]);
                    if (RES) nst[q] = nn[q] + a_dt * Kn;
                } else {
                    C nw = fma2s(w_dt, K, acc[q]);
                    if (NOISE) {
                        const uint4 wd = noise_words(a.seed, blockIdx.x, step, (uint32_t)c);
                        const T nt = RES ? nn[q] : T(0);          // reservoir at the start of the step
                        nw = add2(nw, noise_increment_sfu(wd.x, wd.y, k.sig2 * (T(2) * k.hgc + k.Rr * nt)));
                    }
                    psi[q] = nw;
                    if (RES) nn[q] = nacc[q] + w_dt * Kn;
                    out[c] = nw;                                  // stage-1 input of the next step
                }
            }
        }
        __syncthreads();
    };

    for (int it = 0; it < a.n_steps; ++it) {
        const uint64_t step = a.step0 + (uint64_t)it;
        stage(buf0, buf1, std::integral_constant<int, 1>(), step);
        stage(buf1, buf0, std::integral_constant<int, 2>(), step);
        stage(buf0, buf1, std::integral_constant<int, 3>(), step);
        stage(buf1, buf0, std::integral_constant<int, 4>(), step);
    }

#pragma unroll
    for (int q = 0; q < CPT; ++q) {
        const int c = tid + q * RES_NT;
        if (c < N) {
            psi_g[c] = psi[q];
            if (RES) n_g[c] = nn[q];
        }
    }
    if (blockIdx.x == 0 && tid == 0) {
        a.step_slots[0] = a.step0 + (uint64_t)a.n_steps;
        a.step_slots[1] = a.step0 + (uint64_t)a.n_steps;
    }
}


// ---- cluster form ------------------------------------------------------------------------------------------------------
// Local layout of a stage buffer in the CTA of cluster rank r (rl = ny / cluster rows): row 0 = halo (grid row r*rl - 1),
// rows 1 .. rl = the slab, row rl + 1 = halo (grid row (r+1)*rl), then one cell that stays 0 (a zero boundary in x).
template <typename T, bool RES, bool NOISE, int CPT>
__global__ void __launch_bounds__(RES_NT, 1)
resident_cluster_kernel(const __grid_constant__ ResidentArgs<T> a) {
    namespace cg = cooperative_groups;
    using C = typename Cx<T>::type;
    extern __shared__ __align__(16) unsigned char smem[];
    cg::cluster_group cluster = cg::this_cluster();
    const Geom& g = a.geo;
    const Coef<T>& k = a.k;
    const int ncta = (int)cluster.num_blocks(), rank = (int)cluster.block_rank();
    const int nx = g.nx, rl = g.ny / ncta, NL = rl * nx, NB = (rl + 2) * nx;     // NB = index of the zero cell
    C* buf0 = reinterpret_cast<C*>(smem);
    C* buf1 = buf0 + (NB + 1);
    ushort2* nbr = reinterpret_cast<ushort2*>(buf1 + (NB + 1));                   // west, east (south / north are -+ nx)
    T* Vs = reinterpret_cast<T*>((reinterpret_cast<uintptr_t>(nbr + NL) + 15) & ~(uintptr_t)15);      // (an odd cell count: keep T aligned)
    T* Ps = Vs + NL;

    const int tid = threadIdx.x, nt = blockDim.x;      // (a slab smaller than the largest CTA runs with fewer threads)
    const int real = blockIdx.x / ncta;
    const size_t boff = (size_t)real * g.plane;
    C* psi_g = a.psi + boff;
    T* n_g = RES ? a.n + boff : nullptr;
    const C czero = mk<T>(T(0), T(0));
    const int j0 = rank * rl;                                  // first grid row of the slab
    // neighbours in y: the CTA holding the row below / above the slab (none beyond a zero boundary)
    const bool has_s = !(g.bc_y && rank == 0), has_n = !(g.bc_y && rank == ncta - 1);
    const int rank_s = rank == 0 ? ncta - 1 : rank - 1, rank_n = rank == ncta - 1 ? 0 : rank + 1;
    C* rs0 = cluster.map_shared_rank(buf0, rank_s); C* rs1 = cluster.map_shared_rank(buf1, rank_s);
    C* rn0 = cluster.map_shared_rank(buf0, rank_n); C* rn1 = cluster.map_shared_rank(buf1, rank_n);

    for (int c = tid; c < NB + 1; c += nt) { buf0[c] = czero; buf1[c] = czero; }
    __syncthreads();
    C psi[CPT], acc[CPT];
    T nn[CPT], nacc[CPT], nst[CPT];
#pragma unroll
    for (int q = 0; q < CPT; ++q) {
        const int c = tid + q * nt;
        psi[q] = czero; acc[q] = czero; nn[q] = T(0); nacc[q] = T(0); nst[q] = T(0);
        if (c < NL) {
            const int lr = c / nx, i = c - lr * nx, b = (lr + 1) * nx + i;
            ushort2 nb;
            nb.x = (unsigned short)(i > 0 ? b - 1 : (g.bc_x ? NB : b + nx - 1));
            nb.y = (unsigned short)(i < nx - 1 ? b + 1 : (g.bc_x ? NB : b - nx + 1));
            nbr[c] = nb;
            const size_t gc = (size_t)(j0 + lr) * nx + i;
            Vs[c] = a.V ? a.V[gc] : T(0);
            Ps[c] = (RES && a.P) ? a.P[gc] : T(0);
            psi[q] = psi_g[gc];
            if (RES) nn[q] = n_g[gc];
            buf0[b] = psi[q];
        }
    }
    // halo rows of the first stage input, from global memory
    for (int i = tid; i < nx; i += nt) {
        if (has_s) buf0[i] = psi_g[(size_t)(j0 == 0 ? g.ny - 1 : j0 - 1) * nx + i];
        if (has_n) buf0[(rl + 1) * nx + i] = psi_g[(size_t)(j0 + rl == g.ny ? 0 : j0 + rl) * nx + i];
    }
    cluster.sync();

    auto stage = [&](const C* in, C* out, C* out_s, C* out_n, auto stage_no, const uint64_t step) {
        constexpr int s = decltype(stage_no)::value;
        const T a_dt = s == 3 ? k.dt : k.hdt;
        const T w_dt = (s == 1 || s == 4) ? k.dt6 : k.dt3;
#pragma unroll
        for (int q = 0; q < CPT; ++q) {
            const int c = tid + q * nt;
            if (c < NL) {
                const int lr = c / nx, i = c - lr * nx, b = (lr + 1) * nx + i;
                const ushort2 nb = nbr[c];
                Nbhd<T> h;
                h.c = s == 1 ? psi[q] : in[b];
                h.w = in[nb.x]; h.e = in[nb.y]; h.s = in[b - nx]; h.n = in[b + nx];
                Diff<T> df;
                differences<T, false, false>(k, h, df);
                const T nres = RES ? (s == 1 ? nn[q] : nst[q]) : T(0);
                T Kn;
                const C K = deriv<T, false, RES, false>(k, h.c, df, czero, df, true, nres, Vs[c], Ps[c], czero, czero, Kn);
                if (s == 1) {
                    acc[q] = fma2s(w_dt, K, psi[q]);
                    if (RES) nacc[q] = nn[q] + w_dt * Kn;
                } else if (s < 4) {
                    acc[q] = fma2s(w_dt, K, acc[q]);
                    if (RES) nacc[q] += w_dt * Kn;
                }
                C y;
                if (s < 4) {
                    y = fma2s(a_dt, K, psi[q]);
                    if (RES) nst[q] = nn[q] + a_dt * Kn;
                } else {
                    y = fma2s(w_dt, K, acc[q]);
                    if (NOISE) {
                        const uint4 wd = noise_words(a.seed, (uint32_t)real, step, (uint32_t)((j0 + lr) * nx + i));
                        const T nt = RES ? nn[q] : T(0);          // reservoir at the start of the step
                        y = add2(y, noise_increment_sfu(wd.x, wd.y, k.sig2 * (T(2) * k.hgc + k.Rr * nt)));
                    }
                    psi[q] = y;
                    if (RES) nn[q] = nacc[q] + w_dt * Kn;
                }
                out[b] = y;
                // the slab's first row is the northern halo of the CTA below, its last row the southern halo of the CTA above
                if (lr == 0 && has_s) out_s[(rl + 1) * nx + i] = y;
                if (lr == rl - 1 && has_n) out_n[i] = y;
            }
        }
        cluster.sync();
    };

    for (int it = 0; it < a.n_steps; ++it) {
        const uint64_t step = a.step0 + (uint64_t)it;
        stage(buf0, buf1, rs1, rn1, std::integral_constant<int, 1>(), step);
        stage(buf1, buf0, rs0, rn0, std::integral_constant<int, 2>(), step);
        stage(buf0, buf1, rs1, rn1, std::integral_constant<int, 3>(), step);
        stage(buf1, buf0, rs0, rn0, std::integral_constant<int, 4>(), step);
    }

#pragma unroll
    for (int q = 0; q < CPT; ++q) {
        const int c = tid + q * nt;
        if (c < NL) {
            const int lr = c / nx, i = c - lr * nx;
            const size_t gc = (size_t)(j0 + lr) * nx + i;
            psi_g[gc] = psi[q];
            if (RES) n_g[gc] = nn[q];
        }
    }
    if (blockIdx.x == 0 && tid == 0) {
        a.step_slots[0] = a.step0 + (uint64_t)a.n_steps;
        a.step_slots[1] = a.step0 + (uint64_t)a.n_steps;
    }
}

size_t resident_cluster_smem_bytes(int nx, int rl, int prec64) {
    const size_t rb = prec64 ? 8 : 4, nb = (size_t)(rl + 2) * nx + 1, nl = (size_t)rl * nx;
    return 2 * nb * 2 * rb + nl * sizeof(ushort2) + 2 * nl * rb + 16;      // (+ alignment slack)
}

// Cluster size for one realisation of an nx x ny grid (0 = the cluster form does not apply): the largest of 16, 8, 4, 2 that
// divides ny, gives every CTA at least 2 rows, and whose slab fits 4 cells per thread and the shared memory.
int resident_cluster_size(int nx, int ny, int prec64, bool res) {
    (void)res;
    for (int n = PHX_RESIDENT_MAX_CLUSTER; n >= 2; n >>= 1) {
        if (ny % n != 0 || ny / n < 2) continue;
        const int rl = ny / n;
        if ((size_t)rl * nx > 4u * RES_NT || (size_t)(rl + 2) * nx + 1 > 65535u) continue;
        if (resident_cluster_smem_bytes(nx, rl, prec64) > 200 * 1024) continue;
        return n;
    }
    return 0;
}

template <typename T, bool RES, bool NOISE, int CPT>
static cudaError_t launch_cluster_one(const ResidentArgs<T>& a, int ncta, cudaStream_t st) {
    const size_t smem = resident_cluster_smem_bytes(a.geo.nx, a.geo.ny / ncta, sizeof(T) == 8);
    auto kern = resident_cluster_kernel<T, RES, NOISE, CPT>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    if (ncta > 8) {
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
        if (e != cudaSuccess) return e;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(a.geo.batch * ncta));
    const int nl = a.geo.nx * (a.geo.ny / ncta);
    cfg.blockDim = dim3(CPT == 1 ? (unsigned)((nl + 31) / 32 * 32) : (unsigned)RES_NT);   // one cell per thread: no idle warps at the barriers
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)ncta;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, a);
}


// ---- cluster form, two stages per cluster barrier (scalar model) ----------------------------------------------------------
// As resident_cluster_kernel, but every CTA also computes the odd stages (1 and 3) on ONE extra row above and below its slab
// (the paper's shrinking halo, in rows: redundant arithmetic instead of a barrier), so that a cluster barrier
// is needed only after the even stages: two per RK4 step instead of four, with two halo rows exchanged each time.
// Local rows r = -2 .. rl+1 (buffer row r + 2); threads own the cells of rows -1 .. rl ("extended slab"); three stage buffers
// A, B, C rotate so that no CTA writes into a neighbour's buffer that the neighbour may still be reading:
//   S1: A -> B on rows -1 .. rl      __syncthreads      S2: B -> C on rows 0 .. rl-1, edge rows pushed into the neighbours' C
//   cluster barrier
//   S3: C -> B on rows -1 .. rl      __syncthreads      S4: B -> A on rows 0 .. rl-1 (psi(t+dt)), edge rows pushed into A
//   cluster barrier
// DRIVE: coherent drive E(r) exp(-i omega t) at the stage times (reading Q17), E in shared memory.
template <typename T, bool NOISE, bool DRIVE, int CPT>
__global__ void __launch_bounds__(RES_NT, 1)
resident_pair_kernel(const __grid_constant__ ResidentArgs<T> a) {
    namespace cg = cooperative_groups;
    using C = typename Cx<T>::type;
    extern __shared__ __align__(16) unsigned char smem[];
    cg::cluster_group cluster = cg::this_cluster();
    const Geom& g = a.geo;
    const Coef<T>& k = a.k;
    const int ncta = (int)cluster.num_blocks(), rank = (int)cluster.block_rank();
    const int nx = g.nx, ny = g.ny, rl = ny / ncta, NE = (rl + 2) * nx, NB = (rl + 4) * nx;    // NB = index of the zero cell
    C* bufA = reinterpret_cast<C*>(smem);
    C* bufB = bufA + (NB + 1);
    C* bufC = bufB + (NB + 1);
    ushort2* nbr = reinterpret_cast<ushort2*>(bufC + (NB + 1));                   // west, east
    T* Vs = reinterpret_cast<T*>((reinterpret_cast<uintptr_t>(nbr + NE) + 15) & ~(uintptr_t)15);      // (an odd cell count: keep T aligned)
    C* Es = reinterpret_cast<C*>((reinterpret_cast<uintptr_t>(Vs + NE) + 15) & ~(uintptr_t)15);

    const int tid = threadIdx.x, nt = blockDim.x;
    const int real = blockIdx.x / ncta;
    const size_t boff = (size_t)real * g.plane;
    C* psi_g = a.psi + boff;
    const C czero = mk<T>(T(0), T(0));
    const int j0 = rank * rl;
    const bool has_s = !(g.bc_y && rank == 0), has_n = !(g.bc_y && rank == ncta - 1);
    const int rank_s = rank == 0 ? ncta - 1 : rank - 1, rank_n = rank == ncta - 1 ? 0 : rank + 1;
    C* sA = cluster.map_shared_rank(bufA, rank_s); C* sC = cluster.map_shared_rank(bufC, rank_s);
    C* nA = cluster.map_shared_rank(bufA, rank_n); C* nC = cluster.map_shared_rank(bufC, rank_n);
    // global row of local row r (wrapped); -1 = outside a zero boundary
    auto grow = [&](int r) {
        int j = j0 + r;
        if (j < 0 || j >= ny) {
            if (g.bc_y) return -1;
            j = j < 0 ? j + ny : j - ny;
        }
        return j;
    };

    for (int c = tid; c < 3 * (NB + 1); c += nt) bufA[c] = czero;       // (the three buffers are contiguous)
    __syncthreads();
    C psi[CPT], acc[CPT];
    bool own[CPT], live[CPT];       // own: a cell of the slab; live: a cell of the extended slab inside the domain
#pragma unroll
    for (int q = 0; q < CPT; ++q) {
        const int c = tid + q * nt;
        psi[q] = czero; acc[q] = czero; own[q] = false; live[q] = false;
        if (c < NE) {
            const int er = c / nx, i = c - er * nx, b = (er + 1) * nx + i, j = grow(er - 1);
            own[q] = er >= 1 && er <= rl;
            live[q] = j >= 0;
            ushort2 nb;
            nb.x = (unsigned short)(i > 0 ? b - 1 : (g.bc_x ? NB : b + nx - 1));
            nb.y = (unsigned short)(i < nx - 1 ? b + 1 : (g.bc_x ? NB : b - nx + 1));
            nbr[c] = nb;
            Vs[c] = (a.V && j >= 0) ? a.V[(size_t)j * nx + i] : T(0);
            if constexpr (DRIVE) Es[c] = j >= 0 ? a.E[(size_t)j * nx + i] : czero;
            if (j >= 0) { psi[q] = psi_g[(size_t)j * nx + i]; bufA[b] = psi[q]; }
        }
    }
    for (int i = tid; i < nx; i += nt) {        // the outer halo rows -2 and rl+1 of the first stage input
        const int js = grow(-2), jn = grow(rl + 1);
        if (js >= 0) bufA[i] = psi_g[(size_t)js * nx + i];
        if (jn >= 0) bufA[(rl + 3) * nx + i] = psi_g[(size_t)jn * nx + i];
    }
    (void)has_s; (void)has_n;
    cluster.sync();

    auto odd_stage = [&](const C* in, C* out, auto stage_no, const C qd) {          // stages 1 and 3, on the extended slab
        constexpr int s = decltype(stage_no)::value;
        const T a_dt = s == 3 ? k.dt : k.hdt;
        const T w_dt = s == 1 ? k.dt6 : k.dt3;
#pragma unroll
        for (int q = 0; q < CPT; ++q) {
            const int c = tid + q * nt;
            if (c < NE && live[q]) {
                const int er = c / nx, i = c - er * nx, b = (er + 1) * nx + i;
                const ushort2 nb = nbr[c];
                Nbhd<T> h;
                h.c = s == 1 ? psi[q] : in[b];
                h.w = in[nb.x]; h.e = in[nb.y]; h.s = in[b - nx]; h.n = in[b + nx];
                Diff<T> df;
                differences<T, false, false>(k, h, df);
                T Kn;
                const C K = deriv<T, false, false, DRIVE>(k, h.c, df, czero, df, true, T(0), Vs[c], T(0), DRIVE ? Es[c] : czero, qd, Kn);
                if (own[q]) acc[q] = fma2s(w_dt, K, s == 1 ? psi[q] : acc[q]);
                out[b] = fma2s(a_dt, K, psi[q]);
            }
        }
        __syncthreads();
    };
    auto even_stage = [&](const C* in, C* out, C* out_s, C* out_n, auto stage_no, const uint64_t step, const C qd) {   // stages 2 and 4, on the slab
        constexpr int s = decltype(stage_no)::value;
#pragma unroll
        for (int q = 0; q < CPT; ++q) {
            const int c = tid + q * nt;
            if (c < NE && own[q]) {
                const int er = c / nx, i = c - er * nx, b = (er + 1) * nx + i, r = er - 1;
                const ushort2 nb = nbr[c];
                Nbhd<T> h;
                h.c = in[b];
                h.w = in[nb.x]; h.e = in[nb.y]; h.s = in[b - nx]; h.n = in[b + nx];
                Diff<T> df;
                differences<T, false, false>(k, h, df);
                T Kn;
                const C K = deriv<T, false, false, DRIVE>(k, h.c, df, czero, df, true, T(0), Vs[c], T(0), DRIVE ? Es[c] : czero, qd, Kn);
                C y;
                if (s == 2) {
                    acc[q] = fma2s(k.dt3, K, acc[q]);
                    y = fma2s(k.hdt, K, psi[q]);
                } else {
                    y = fma2s(k.dt6, K, acc[q]);
                    if (NOISE) {
                        const uint4 wd = noise_words(a.seed, (uint32_t)real, step, (uint32_t)((j0 + r) * nx + i));
                        y = add2(y, noise_increment_sfu(wd.x, wd.y, k.sig2 * (T(2) * k.hgc)));
                    }
                    psi[q] = y;
                }
                out[b] = y;
                // the two first rows of the slab are rows rl, rl+1 of the CTA below; the two last rows are rows -2, -1 of the CTA above
                if (r < 2 && has_s) out_s[(rl + r + 2) * nx + i] = y;
                if (r >= rl - 2 && has_n) out_n[(r - rl + 2) * nx + i] = y;
            }
        }
        cluster.sync();
    };

    for (int it = 0; it < a.n_steps; ++it) {
        const uint64_t step = a.step0 + (uint64_t)it;
        if (it > 0) {           // the cells of the extra rows take psi(t) from what the neighbours pushed
#pragma unroll
            for (int q = 0; q < CPT; ++q) {
                const int c = tid + q * nt;
                if (c < NE && live[q] && !own[q]) psi[q] = bufA[(c / nx + 1) * nx + c % nx];
            }
        }
        C q1 = czero, q23 = czero, q4 = czero;          // (1/hbar) exp(-i omega t_s) at t, t + dt/2, t + dt, phase in double
        if constexpr (DRIVE) {
            auto phase = [&](double cs) {
                double sn, cn;
                sincos(-k.omega * (((double)step + cs) * k.dt_d), &sn, &cn);
                return mk<T>(k.ih * (T)cn, k.ih * (T)sn);
            };
            q1 = phase(0.0); q23 = phase(0.5); q4 = phase(1.0);
        }
        odd_stage(bufA, bufB, std::integral_constant<int, 1>(), q1);
        even_stage(bufB, bufC, sC, nC, std::integral_constant<int, 2>(), step, q23);
        odd_stage(bufC, bufB, std::integral_constant<int, 3>(), q23);
        even_stage(bufB, bufA, sA, nA, std::integral_constant<int, 4>(), step, q4);
    }

#pragma unroll
    for (int q = 0; q < CPT; ++q) {
        const int c = tid + q * nt;
        if (c < NE && own[q]) {
            const int er = c / nx, i = c - er * nx;
            psi_g[(size_t)(j0 + er - 1) * nx + i] = psi[q];
        }
    }
    if (blockIdx.x == 0 && tid == 0) {
        a.step_slots[0] = a.step0 + (uint64_t)a.n_steps;
        a.step_slots[1] = a.step0 + (uint64_t)a.n_steps;
    }
}

size_t resident_pair_smem_bytes(int nx, int rl, int prec64, bool drive = true) {
    const size_t rb = prec64 ? 8 : 4, nb = (size_t)(rl + 4) * nx + 1, ne = (size_t)(rl + 2) * nx;
    return 3 * nb * 2 * rb + ne * sizeof(ushort2) + ne * rb + (drive ? ne * 2 * rb : 0) + 48;      // (+ alignment slack)
}

// The pair kernel applies to the scalar model when the extended slab fits 4 cells per thread.
bool resident_pair_ok(int nx, int ny, int ncta, int prec64) {
    if (ncta < 2 || ny % ncta != 0) return false;
    const int rl = ny / ncta;
    if (rl < 2 || (size_t)(rl + 2) * nx > 4u * RES_NT || (size_t)(rl + 4) * nx + 1 > 65535u) return false;
    return resident_pair_smem_bytes(nx, rl, prec64) <= 200 * 1024;
}

template <typename T, bool NOISE, bool DRIVE, int CPT>
static cudaError_t launch_pair_one(const ResidentArgs<T>& a, int ncta, cudaStream_t st) {
    const int rl = a.geo.ny / ncta, ne = (rl + 2) * a.geo.nx;
    const size_t smem = resident_pair_smem_bytes(a.geo.nx, rl, sizeof(T) == 8, DRIVE);
    auto kern = resident_pair_kernel<T, NOISE, DRIVE, CPT>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    if (ncta > 8) {
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
        if (e != cudaSuccess) return e;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(a.geo.batch * ncta));
    cfg.blockDim = dim3(CPT == 1 ? (unsigned)((ne + 31) / 32 * 32) : (unsigned)RES_NT);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)ncta;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, a);
}

template <typename T>
static cudaError_t launch_pair_t(const ResidentArgs<T>& a, bool noise, int ncta, cudaStream_t st) {
    const int need = ((a.geo.ny / ncta + 2) * a.geo.nx + RES_NT - 1) / RES_NT;
    if (a.E) {
        if (noise) return need == 1 ? launch_pair_one<T, true, true, 1>(a, ncta, st) : launch_pair_one<T, true, true, 4>(a, ncta, st);
        return need == 1 ? launch_pair_one<T, false, true, 1>(a, ncta, st) : launch_pair_one<T, false, true, 4>(a, ncta, st);
    }
    if (noise) return need == 1 ? launch_pair_one<T, true, false, 1>(a, ncta, st) : launch_pair_one<T, true, false, 4>(a, ncta, st);
    return need == 1 ? launch_pair_one<T, false, false, 1>(a, ncta, st) : launch_pair_one<T, false, false, 4>(a, ncta, st);
}

template <typename T>
static cudaError_t launch_cluster_t(const ResidentArgs<T>& a, bool res, bool noise, cudaStream_t st) {
    const int ncta = resident_cluster_size(a.geo.nx, a.geo.ny, sizeof(T) == 8, res);
    if (ncta == 0) return cudaErrorInvalidConfiguration;
    if (PHX_RESIDENT_PAIR && !res && resident_pair_ok(a.geo.nx, a.geo.ny, ncta, sizeof(T) == 8)) return launch_pair_t<T>(a, noise, ncta, st);
    if (a.E) return cudaErrorInvalidConfiguration;          // (a drive: the pair kernel only)
    const int need = (a.geo.nx * (a.geo.ny / ncta) + RES_NT - 1) / RES_NT;
#define PHX_RESC_CASE(R, NZ)                                                  \
    if (res == R && noise == NZ) {                                            \
        if (need == 1) return launch_cluster_one<T, R, NZ, 1>(a, ncta, st);   \
        return launch_cluster_one<T, R, NZ, 4>(a, ncta, st);                  \
    }
    PHX_RESC_CASE(false, false)
    PHX_RESC_CASE(false, true)
    PHX_RESC_CASE(true, false)
    PHX_RESC_CASE(true, true)
#undef PHX_RESC_CASE
    return cudaErrorInvalidConfiguration;
}

// A driven scalar grid can run variant RESIDENT iff the pair kernel applies to it.
bool resident_drive_ok(int nx, int ny, int prec64) {
    const int ncta = resident_cluster_size(nx, ny, prec64, false);
    return PHX_RESIDENT_PAIR && ncta != 0 && resident_pair_ok(nx, ny, ncta, prec64);
}

cudaError_t launch_resident_cluster_32(const ResidentArgs<float>& a, bool res, bool noise, cudaStream_t st) { return launch_cluster_t<float>(a, res, noise, st); }
cudaError_t launch_resident_cluster_64(const ResidentArgs<double>& a, bool res, bool noise, cudaStream_t st) { return launch_cluster_t<double>(a, res, noise, st); }

size_t resident_smem_bytes(int cells, int prec64) {
    const size_t rb = prec64 ? 8 : 4;
    return 2 * (size_t)(cells + 1) * 2 * rb + (size_t)cells * sizeof(ushort4) + 2 * (size_t)cells * rb;
}

// Cells per thread the instantiations cover (0 = the grid does not fit this variant).
int resident_cpt(size_t cells, int prec64, bool res) {
    if (cells > 65534) return 0;                      // neighbour indices are 16 bit
    const int max_cpt = (prec64 && res) ? 4 : 8;      // register budget of 128 per thread
    const int need = ((int)cells + RES_NT - 1) / RES_NT;
    if (need > max_cpt) return 0;
    if (resident_smem_bytes((int)cells, prec64) > 227 * 1024) return 0;
    return need <= 4 ? 4 : 8;
}

template <typename T, bool RES, bool NOISE, int CPT>
static cudaError_t launch_one(const ResidentArgs<T>& a, cudaStream_t st) {
    const size_t smem = resident_smem_bytes(a.geo.nx * a.geo.ny, sizeof(T) == 8);
    auto kern = resident_kernel<T, RES, NOISE, CPT>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    kern<<<a.geo.batch, RES_NT, smem, st>>>(a);
    return cudaGetLastError();
}

template <typename T>
static cudaError_t launch_t(const ResidentArgs<T>& a, bool res, bool noise, cudaStream_t st) {
    const int cpt = resident_cpt((size_t)a.geo.nx * (size_t)a.geo.ny, sizeof(T) == 8, res);
    if (cpt == 0) return cudaErrorInvalidConfiguration;
#define PHX_RES_CASE(R, NZ)                                                      \
    if (res == R && noise == NZ) {                                               \
        if (cpt == 4) return launch_one<T, R, NZ, 4>(a, st);                     \
        if constexpr (!(R && sizeof(T) == 8)) return launch_one<T, R, NZ, 8>(a, st); \
    }
    PHX_RES_CASE(false, false)
    PHX_RES_CASE(false, true)
    PHX_RES_CASE(true, false)
    PHX_RES_CASE(true, true)
#undef PHX_RES_CASE
    return cudaErrorInvalidConfiguration;
}

cudaError_t launch_resident_32(const ResidentArgs<float>& a, bool res, bool noise, cudaStream_t st) { return launch_t<float>(a, res, noise, st); }
cudaError_t launch_resident_64(const ResidentArgs<double>& a, bool res, bool noise, cudaStream_t st) { return launch_t<double>(a, res, noise, st); }

}  // namespace phx
