// sn_levelset.cu -- level-set re-initialisation (include/sn_levelset.h).
// PAPER.md:131-141 (section 2.2, eqs. 6-7); readings L1..L6 in DESIGN.md section 3.  Three kernels:
//   k_ls_crossings  every node tests its +x and +y grid edge for a sign change and appends the linearly interpolated
//                   front position to a list (warp-aggregated atomic append; the order of the list is irrelevant
//                   because only an exact minimum is taken over it);
//   k_ls_distance   the paper's "distances of all grid points to the flame front positions are compared": nodes x
//                   crossings pairs, crossings staged through shared memory in chunks and broadcast to the threads,
//                   4 nodes per thread in registers; the crossing list is also split across CTAs (grid.y) so that any
//                   problem size fills the 148 SMs, partial minima merged with atomicMin on the bit pattern of the
//                   non-negative squared distance (exact, order-independent);
//   k_ls_blend      d = copysign(sqrt(min), S_old), H(|d|), eq. (6).
// Bound: plain fp64 ALU work (5 fp64 instructions per node-crossing pair); no tensor cores (not a contraction).
#include "../../include/sn_levelset.h"

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <string>

#include <cuda_runtime.h>

namespace {

thread_local std::string g_ls_err;

void ls_err(const char* fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    g_ls_err = buf;
}

#define LS_TRY(expr)                                                                        \
    do {                                                                                    \
        cudaError_t e__ = (expr);                                                           \
        if (e__ != cudaSuccess) {                                                           \
            ls_err("%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e__), __FILE__, __LINE__); \
            return -2;                                                                      \
        }                                                                                   \
    } while (0)

constexpr int kLsThreads = 256;      // threads per CTA of the distance kernel
constexpr int kLsNpt = 4;            // nodes per thread
constexpr int kLsChunk = 1024;       // crossings per shared-memory chunk (16 KB)

// L2 / L3: edges (i,j)-(i+1,j) and (i,j)-(i,j+1); cut when one end is < 0 and the other >= 0.
__global__ void __launch_bounds__(256) k_ls_crossings(int nx, int ny, double dr, double dz, const double* __restrict__ S,
                                                      double2* __restrict__ cross, unsigned int* __restrict__ count) {
    const size_t n = (size_t)nx * ny;
    const int lane = threadIdx.x & 31;
    for (size_t base = (size_t)blockIdx.x * blockDim.x; base < n; base += (size_t)gridDim.x * blockDim.x) {
        const size_t idx = base + threadIdx.x;
        double2 c[2];
        int m = 0;
        if (idx < n) {
            const int j = (int)(idx / nx), i = (int)(idx - (size_t)j * nx);
            const double sa = S[idx];
            const double xa = __dmul_rn((double)i, dr), ya = __dmul_rn((double)j, dz);
            if (i + 1 < nx) {
                const double sb = S[idx + 1];
                if ((sa < 0.0) != (sb < 0.0)) c[m++] = make_double2(__fma_rn(__ddiv_rn(sa, __dsub_rn(sa, sb)), dr, xa), ya);
            }
            if (j + 1 < ny) {
                const double sb = S[idx + nx];
                if ((sa < 0.0) != (sb < 0.0)) c[m++] = make_double2(xa, __fma_rn(__ddiv_rn(sa, __dsub_rn(sa, sb)), dz, ya));
            }
        }
        // warp-aggregated append: one atomic per warp
        int pre = m;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, pre, o);
            if (lane >= o) pre += t;
        }
        const int total = __shfl_sync(0xffffffffu, pre, 31);
        unsigned int at = 0;
        if (lane == 31 && total > 0) at = atomicAdd(count, (unsigned int)total);
        at = __shfl_sync(0xffffffffu, at, 31);
        for (int k = 0; k < m; ++k) cross[at + (pre - m) + k] = c[k];
    }
}

// grid = (node tiles of kLsThreads * kLsNpt nodes, splits of the crossing list).
__global__ void __launch_bounds__(kLsThreads) k_ls_distance(int nx, int ny, double dr, double dz,
                                                            const double2* __restrict__ cross, unsigned int ncross,
                                                            unsigned long long* __restrict__ d2) {
    __shared__ double2 sc[kLsChunk];
    const size_t n = (size_t)nx * ny;
    const unsigned int per = (ncross + gridDim.y - 1) / gridDim.y;
    const unsigned int c0 = blockIdx.y * per, c1 = min(ncross, c0 + per);
    double x[kLsNpt], y[kLsNpt], best[kLsNpt];
    size_t node[kLsNpt];
#pragma unroll
    for (int k = 0; k < kLsNpt; ++k) {
        node[k] = ((size_t)blockIdx.x * kLsNpt + k) * kLsThreads + threadIdx.x;
        const size_t q = node[k] < n ? node[k] : n - 1;
        const int j = (int)(q / nx), i = (int)(q - (size_t)j * nx);
        x[k] = __dmul_rn((double)i, dr);
        y[k] = __dmul_rn((double)j, dz);
        best[k] = INFINITY;
    }
    for (unsigned int base = c0; base < c1; base += kLsChunk) {
        const int m = (int)min((unsigned int)kLsChunk, c1 - base);
        for (int t = threadIdx.x; t < m; t += kLsThreads) sc[t] = cross[base + t];
        __syncthreads();
#pragma unroll 4
        for (int c = 0; c < m; ++c) {
            const double2 p = sc[c];                     // broadcast
#pragma unroll
            for (int k = 0; k < kLsNpt; ++k) {
                const double dx = __dsub_rn(x[k], p.x), dy = __dsub_rn(y[k], p.y);
                const double dd = __fma_rn(dy, dy, __dmul_rn(dx, dx));
                best[k] = dd < best[k] ? dd : best[k];
            }
        }
        __syncthreads();
    }
#pragma unroll
    for (int k = 0; k < kLsNpt; ++k)
        if (node[k] < n) atomicMin(d2 + node[k], (unsigned long long)__double_as_longlong(best[k]));   // dd >= 0: bits order like values
}

// L4 / L5 and eqs. (6)-(7).
__global__ void __launch_bounds__(256) k_ls_blend(size_t n, double delta, const double* __restrict__ S_old,
                                                  const unsigned long long* __restrict__ d2, double* __restrict__ S_new,
                                                  double* __restrict__ dist) {
    const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= n) return;
    const double so = S_old[idx];
    const double dmin = __dsqrt_rn(__longlong_as_double((long long)d2[idx]));
    const double d = copysign(dmin, so);
    const double d0 = __dmul_rn(3.0, delta), w = __ddiv_rn(delta, 3.0);
    const double h = __ddiv_rn(__dsub_rn(1.0, tanh(__ddiv_rn(__dsub_rn(dmin, d0), w))),
                               __dsub_rn(1.0, tanh(__ddiv_rn(-d0, w))));
    S_new[idx] = __dadd_rn(__dmul_rn(h, so), __dmul_rn(__dsub_rn(1.0, h), d));
    if (dist) dist[idx] = d;
}

// L6: no crossing anywhere -- S unchanged, d = copysign(inf, S_old)
__global__ void __launch_bounds__(256) k_ls_nocross(size_t n, const double* __restrict__ S_old, double* __restrict__ S_new,
                                                    double* __restrict__ dist) {
    const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= n) return;
    const double so = S_old[idx];
    S_new[idx] = so;
    if (dist) dist[idx] = copysign(INFINITY, so);
}

}  // namespace

struct sn_levelset {
    int nx = 0, ny = 0, device = 0, num_sms = 0;
    double dr = 0, dz = 0, delta = 0;
    double2* d_cross = nullptr;
    unsigned long long* d_d2 = nullptr;
    unsigned int* d_count = nullptr;
    unsigned int* h_count = nullptr;          // pinned
    double *d_in = nullptr, *d_out = nullptr, *d_dist = nullptr;   // staging of the host entry point
    cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
    double st_cross = 0, st_pairs = 0, st_dist_ms = 0, st_total_ms = 0, st_launches = 0;
};

extern "C" {

const char* sn_levelset_last_error(void) { return g_ls_err.c_str(); }

sn_levelset* sn_levelset_create(int nx, int ny, double dr, double dz, double delta) {
    g_ls_err.clear();
    if (nx < 2 || ny < 2) { ls_err("nx, ny must be >= 2"); return nullptr; }
    if (!(dr > 0) || !(dz > 0) || !(delta > 0) || !std::isfinite(dr) || !std::isfinite(dz) || !std::isfinite(delta)) {
        ls_err("dr, dz, delta must be finite and > 0");
        return nullptr;
    }
    if ((long long)nx * ny > (1ll << 30)) { ls_err("grid too large"); return nullptr; }
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
        ls_err("no CUDA device: %s", cudaGetErrorString(cudaGetLastError()));
        return nullptr;
    }
    if (prop.major != 10) {
        ls_err("device %d is sm_%d%d; this library is built for sm_100a only (no fallback)", dev, prop.major, prop.minor);
        return nullptr;
    }
    sn_levelset* h = new (std::nothrow) sn_levelset();
    if (!h) { ls_err("out of host memory"); return nullptr; }
    h->nx = nx; h->ny = ny; h->dr = dr; h->dz = dz; h->delta = delta; h->device = dev;
    h->num_sms = prop.multiProcessorCount;
    const size_t n = (size_t)nx * ny;
    bool ok = cudaMalloc((void**)&h->d_cross, sizeof(double2) * 2 * n) == cudaSuccess &&
              cudaMalloc((void**)&h->d_d2, sizeof(unsigned long long) * n) == cudaSuccess &&
              cudaMalloc((void**)&h->d_count, sizeof(unsigned int)) == cudaSuccess &&
              cudaMallocHost((void**)&h->h_count, sizeof(unsigned int)) == cudaSuccess;
    for (auto& e : h->ev) ok = ok && cudaEventCreate(&e) == cudaSuccess;
    if (!ok) {
        ls_err("CUDA allocation failed: %s", cudaGetErrorString(cudaGetLastError()));
        sn_levelset_destroy(h);
        return nullptr;
    }
    return h;
}

void sn_levelset_destroy(sn_levelset* h) {
    if (!h) return;
    cudaFree(h->d_cross); cudaFree(h->d_d2); cudaFree(h->d_count);
    cudaFree(h->d_in); cudaFree(h->d_out); cudaFree(h->d_dist);
    if (h->h_count) cudaFreeHost(h->h_count);
    for (auto& e : h->ev) if (e) cudaEventDestroy(e);
    delete h;
}

int64_t sn_levelset_reinit(sn_levelset* h, const double* S_old, double* S_new, double* dist, void* stream) {
    g_ls_err.clear();
    if (!h || !S_old || !S_new) { ls_err("NULL argument"); return -1; }
    if (S_old == S_new || S_old == dist) { ls_err("S_new / dist must not alias S_old"); return -1; }
    cudaStream_t st = (cudaStream_t)stream;
    LS_TRY(cudaSetDevice(h->device));
    const size_t n = (size_t)h->nx * h->ny;
    LS_TRY(cudaEventRecord(h->ev[0], st));
    LS_TRY(cudaMemsetAsync(h->d_count, 0, sizeof(unsigned int), st));
    LS_TRY(cudaMemsetAsync(h->d_d2, 0x7f, sizeof(unsigned long long) * n, st));     // 0x7f7f... = 1.4e306: "no crossing yet"
    const int gx = (int)std::min<size_t>((n + 255) / 256, (size_t)h->num_sms * 8);
    k_ls_crossings<<<gx, 256, 0, st>>>(h->nx, h->ny, h->dr, h->dz, S_old, h->d_cross, h->d_count);
    LS_TRY(cudaGetLastError());
    LS_TRY(cudaMemcpyAsync(h->h_count, h->d_count, sizeof(unsigned int), cudaMemcpyDeviceToHost, st));
    LS_TRY(cudaStreamSynchronize(st));                    // the crossing count sizes the next launch
    const unsigned int nc = *h->h_count;
    h->st_launches = 1;
    h->st_cross = nc;
    h->st_pairs = (double)nc * (double)n;
    h->st_dist_ms = 0;
    if (nc == 0) {                                        // L6: nothing to measure distances to
        k_ls_nocross<<<(unsigned int)((n + 255) / 256), 256, 0, st>>>(n, S_old, S_new, dist);
        LS_TRY(cudaGetLastError());
        h->st_launches = 2;
        LS_TRY(cudaEventRecord(h->ev[3], st));
        LS_TRY(cudaStreamSynchronize(st));
        float ms = 0;
        LS_TRY(cudaEventElapsedTime(&ms, h->ev[0], h->ev[3]));
        h->st_total_ms = ms;
        return 0;
    }
    const unsigned int tiles = (unsigned int)((n + kLsThreads * kLsNpt - 1) / (kLsThreads * kLsNpt));
    unsigned int splits = (4u * (unsigned int)h->num_sms + tiles - 1) / tiles;
    const unsigned int max_splits = (nc + 255) / 256;
    if (splits > max_splits) splits = max_splits;
    if (splits < 1) splits = 1;
    if (splits > 65535) splits = 65535;
    LS_TRY(cudaEventRecord(h->ev[1], st));
    k_ls_distance<<<dim3(tiles, splits), kLsThreads, 0, st>>>(h->nx, h->ny, h->dr, h->dz, h->d_cross, nc, h->d_d2);
    LS_TRY(cudaGetLastError());
    LS_TRY(cudaEventRecord(h->ev[2], st));
    k_ls_blend<<<(unsigned int)((n + 255) / 256), 256, 0, st>>>(n, h->delta, S_old, h->d_d2, S_new, dist);
    LS_TRY(cudaGetLastError());
    LS_TRY(cudaEventRecord(h->ev[3], st));
    LS_TRY(cudaStreamSynchronize(st));
    float ms = 0;
    LS_TRY(cudaEventElapsedTime(&ms, h->ev[1], h->ev[2]));
    h->st_dist_ms = ms;
    LS_TRY(cudaEventElapsedTime(&ms, h->ev[0], h->ev[3]));
    h->st_total_ms = ms;
    h->st_launches = 3;
    return (int64_t)nc;
}

int64_t sn_levelset_reinit_host(sn_levelset* h, const double* S_old_host, double* S_new_host, double* dist_host,
                                void* stream) {
    g_ls_err.clear();
    if (!h || !S_old_host || !S_new_host) { ls_err("NULL argument"); return -1; }
    cudaStream_t st = (cudaStream_t)stream;
    LS_TRY(cudaSetDevice(h->device));
    const size_t bytes = sizeof(double) * (size_t)h->nx * h->ny;
    if (!h->d_in) {
        LS_TRY(cudaMalloc((void**)&h->d_in, bytes));
        LS_TRY(cudaMalloc((void**)&h->d_out, bytes));
        LS_TRY(cudaMalloc((void**)&h->d_dist, bytes));
    }
    LS_TRY(cudaMemcpyAsync(h->d_in, S_old_host, bytes, cudaMemcpyHostToDevice, st));
    const int64_t rc = sn_levelset_reinit(h, h->d_in, h->d_out, dist_host ? h->d_dist : nullptr, st);
    if (rc < 0) return rc;
    LS_TRY(cudaMemcpyAsync(S_new_host, h->d_out, bytes, cudaMemcpyDeviceToHost, st));
    if (dist_host) LS_TRY(cudaMemcpyAsync(dist_host, h->d_dist, bytes, cudaMemcpyDeviceToHost, st));
    LS_TRY(cudaStreamSynchronize(st));
    return rc;
}

int sn_levelset_get_stat(sn_levelset* h, const char* key, double* out) {
    g_ls_err.clear();
    if (!h || !key || !out) { ls_err("NULL argument"); return -1; }
    if (!strcmp(key, "crossings")) { *out = h->st_cross; return 0; }
    if (!strcmp(key, "pairs")) { *out = h->st_pairs; return 0; }
    if (!strcmp(key, "distance_ms")) { *out = h->st_dist_ms; return 0; }
    if (!strcmp(key, "total_ms")) { *out = h->st_total_ms; return 0; }
    if (!strcmp(key, "launches")) { *out = h->st_launches; return 0; }
    ls_err("unknown stat '%s'", key);
    return -1;
}

}  // extern "C"
