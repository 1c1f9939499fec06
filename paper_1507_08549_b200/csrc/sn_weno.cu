// sn_weno.cu -- WENO-5 / global Lax-Friedrichs flux reconstruction (include/sn_weno.h).
// PAPER.md:79-89 (eqs. 1-4, left-hand sides), PAPER.md:95 (finite-difference WENO, global LF splitting, upwinded
// reconstruction of both split fluxes), PAPER.md:402 (gamma-law EOS, Courant number 0.5); readings W1..W9 in DESIGN.md.
// Kernels:
//   k_weno_speeds   alpha_r, alpha_z = max over all cells of |v| + c_s: registers -> warp REDUX on the order-preserving
//                   bit pattern -> shared memory -> one atomicMax per CTA (exact, order-independent);
//   k_weno_dt       dt = cfl / (alpha_r/dr + alpha_z/dz) on the device, so that a Runge-Kutta step needs no host round trip;
//   k_weno_rhs      one CTA per 32 x 8 tile: the tile plus its 3-cell halo (ghost cells by index mapping) goes to shared
//                   memory once together with p, v_r, v_z; every thread reconstructs the fluxes through the east and the
//                   north face of its cell (4 components x 2 split fluxes x WENO-5 each); the west / south face values
//                   come from the neighbouring thread (warp shuffle in r, shared memory in z; only the first column /
//                   row of a tile recomputes them); the Runge-Kutta stage update is fused into the epilogue.
// Bound: plain fp64 ALU work (~2.75 k fp64 instructions per cell -- an IEEE division is ~18 of them -- against 64 B of compulsory traffic); no tensor cores
// (not a contraction).  Arithmetic pinned like the rest of the library: -fmad=false, expression trees typed out.
#include "../../include/sn_weno.h"

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <string>

#include <cuda_runtime.h>

namespace {

thread_local std::string g_wn_err;

void wn_err(const char* fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    g_wn_err = buf;
}

#define WN_TRY(expr)                                                                        \
    do {                                                                                    \
        cudaError_t e__ = (expr);                                                           \
        if (e__ != cudaSuccess) {                                                           \
            wn_err("%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e__), __FILE__, __LINE__); \
            return -2;                                                                      \
        }                                                                                   \
    } while (0)

constexpr int kTX = 32, kTY = 8, kHalo = 3;
constexpr int kSX = kTX + 2 * kHalo, kSY = kTY + 2 * kHalo;      // shared tile with halo: 38 x 14

struct WenoGeom {
    int nr, nz;
    double dr, dz, gamma;
    int bc[4];
};

// W7: source cell of position i (any integer) and whether the normal momentum flips.  Positions far outside the grid
// (only touched by the inactive threads of a partial tile) are clamped.
__device__ __forceinline__ int ghost_src(int i, int n, int lo, int hi, bool& flip) {
    flip = false;
    int s = i;
    if (i < 0) {
        if (lo == 0) s = 0;
        else if (lo == 1) { s = -1 - i; flip = true; }
        else s = i + n;
    } else if (i >= n) {
        if (hi == 0) s = n - 1;
        else if (hi == 1) { s = 2 * n - 1 - i; flip = true; }
        else s = i - n;
    }
    return s < 0 ? 0 : s >= n ? n - 1 : s;
}

__device__ __forceinline__ double pressure_of(double gamma, double u0, double u1, double u2, double u3) {
    const double ke = (u1 * u1 + u2 * u2) / (2.0 * u0);                  // W2
    return (gamma - 1.0) * (u3 - ke);
}

// W5: Jiang-Shu WENO-5 value at the downwind face of cell c from (a, b, c, d, e), a on the upwind side
__device__ __forceinline__ double weno5(double a, double b, double c, double d, double e) {
    const double k6 = 1.0 / 6.0;
    const double q0 = (2.0 * a - 7.0 * b + 11.0 * c) * k6;
    const double q1 = (-b + 5.0 * c + 2.0 * d) * k6;
    const double q2 = (2.0 * c + 5.0 * d - e) * k6;
    const double s0 = a - 2.0 * b + c, t0 = a - 4.0 * b + 3.0 * c;
    const double s1 = b - 2.0 * c + d, t1 = b - d;
    const double s2 = c - 2.0 * d + e, t2 = 3.0 * c - 4.0 * d + e;
    const double b0 = (13.0 / 12.0) * (s0 * s0) + 0.25 * (t0 * t0);
    const double b1 = (13.0 / 12.0) * (s1 * s1) + 0.25 * (t1 * t1);
    const double b2 = (13.0 / 12.0) * (s2 * s2) + 0.25 * (t2 * t2);
    const double e0 = 1.0e-6 + b0, e1 = 1.0e-6 + b1, e2 = 1.0e-6 + b2;
    const double a0 = 0.1 / (e0 * e0), a1 = 0.6 / (e1 * e1), a2 = 0.3 / (e2 * e2);
    const double sum = (a0 + a1) + a2;
    return ((a0 * q0 + a1 * q1) + a2 * q2) / sum;
}

__device__ __forceinline__ unsigned long long warp_max_u64(unsigned long long k) {
    const unsigned hi = (unsigned)(k >> 32), lo = (unsigned)k;
    const unsigned mh = __reduce_max_sync(0xffffffffu, hi);
    const unsigned ml = __reduce_max_sync(0xffffffffu, hi == mh ? lo : 0u);
    return ((unsigned long long)mh << 32) | ml;
}

// W4.  alpha[0..1]: bit patterns of non-negative doubles (NaN sorts highest: sticky, like the oracle's), zeroed before.
__global__ void __launch_bounds__(256) k_weno_speeds(WenoGeom g, const double* __restrict__ U,
                                                     unsigned long long* __restrict__ alpha) {
    const size_t n = (size_t)g.nr * g.nz;
    unsigned long long kr = 0ull, kz = 0ull;
    for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (size_t)gridDim.x * blockDim.x) {
        const double u0 = U[k], u1 = U[n + k], u2 = U[2 * n + k], u3 = U[3 * n + k];
        const double c = sqrt(g.gamma * pressure_of(g.gamma, u0, u1, u2, u3) / u0);
        const double sr = fabs(u1 / u0) + c, sz = fabs(u2 / u0) + c;
        const unsigned long long br = (unsigned long long)__double_as_longlong(sr) & 0x7fffffffffffffffull;
        const unsigned long long bz = (unsigned long long)__double_as_longlong(sz) & 0x7fffffffffffffffull;
        kr = br > kr ? br : kr;
        kz = bz > kz ? bz : kz;
    }
    // warp -> CTA -> one atomic pair per CTA (warps hitting the same two words serialise in L2)
    __shared__ unsigned long long sk[2][8];
    kr = warp_max_u64(kr);
    kz = warp_max_u64(kz);
    if ((threadIdx.x & 31) == 0) { sk[0][threadIdx.x >> 5] = kr; sk[1][threadIdx.x >> 5] = kz; }
    __syncthreads();
    if (threadIdx.x < 32) {
        kr = warp_max_u64(threadIdx.x < 8 ? sk[0][threadIdx.x] : 0ull);
        kz = warp_max_u64(threadIdx.x < 8 ? sk[1][threadIdx.x] : 0ull);
        if (threadIdx.x == 0) {
            atomicMax(alpha, kr);
            atomicMax(alpha + 1, kz);
        }
    }
}

// W8: dt = cfl / (alpha_r / dr + alpha_z / dz)
__global__ void k_weno_dt(WenoGeom g, const double* __restrict__ alpha, double cfl, double* __restrict__ dt) {
    if (threadIdx.x == 0 && blockIdx.x == 0) *dt = cfl / (alpha[0] / g.dr + alpha[1] / g.dz);
}

// The step of sn_weno_evolve, decided on the device: the Courant step, shortened if it would pass t_end -- the same
// expressions, in the same order, as the host loop they replace (and as the oracle's march): use = (t_end - t) / dt_full
// * cfl for the last step, dt = use / (alpha_r/dr + alpha_z/dz).  tstate[0] = t (advanced here), tstate[1] = 1 if this
// was the shortened last step.
__global__ void k_weno_dt_evolve(WenoGeom g, const double* __restrict__ alpha, double cfl, double t_end,
                                 double* __restrict__ dt, double* __restrict__ tstate) {
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        const double s = alpha[0] / g.dr + alpha[1] / g.dz;
        const double t = tstate[0];
        const double dt_full = cfl / s;
        const double use = t + dt_full > t_end ? (t_end - t) / dt_full * cfl : cfl;
        const double d = use / s;
        *dt = d;
        tstate[0] = t + d;
        tstate[1] = use != cfl ? 1.0 : 0.0;
    }
}

struct RhsParams {
    WenoGeom g;
    const double* U;         // stage input (stencil source)
    const double* U0;        // MODE 2: state at the start of the step
    double* out;             // MODE 0: L; MODE 1: U + dt L; MODE 2: ca U0 + cb (U + dt L)
    const double* alpha;     // device: alpha_r, alpha_z
    const double* dt;        // device (MODE 1, 2)
    double ca, cb;
};

struct TileSmem {
    double u[4][kSY][kSX];
    double p[kSY][kSX], vr[kSY][kSX], vz[kSY][kSX];
    double gn[4][kTY][kTX];      // north-face fluxes of the tile's cells (z exchange between thread rows)
};

// numerical flux (4 components) through the face between the shared-tile cell (ly, lx) and its + neighbour along DIR
template <int DIR>
__device__ __forceinline__ void face_flux(const TileSmem& s, int ly, int lx, double alpha, double fh[4]) {
    double u[6][4], v[6], p[6];
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        const int y = DIR == 0 ? ly : ly - 2 + k, x = DIR == 0 ? lx - 2 + k : lx;
#pragma unroll
        for (int c = 0; c < 4; ++c) u[k][c] = s.u[c][y][x];
        v[k] = DIR == 0 ? s.vr[y][x] : s.vz[y][x];
        p[k] = s.p[y][x];
    }
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        double fp[6], fm[6];
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            double f;                                                   // W3
            if (c == 0) f = u[k][1 + DIR];
            else if (c == 3) f = (u[k][3] + p[k]) * v[k];
            else {
                f = u[k][c] * v[k];
                if (c == 1 + DIR) f = f + p[k];
            }
            const double au = alpha * u[k][c];
            fp[k] = 0.5 * (f + au);                                     // W4
            fm[k] = 0.5 * (f - au);
        }
        fh[c] = weno5(fp[0], fp[1], fp[2], fp[3], fp[4]) + weno5(fm[5], fm[4], fm[3], fm[2], fm[1]);
    }
}

template <int MODE>
__global__ void __launch_bounds__(kTX* kTY) k_weno_rhs(const RhsParams P) {
    __shared__ TileSmem s;
    const WenoGeom& g = P.g;
    const int tx = threadIdx.x, ty = threadIdx.y, tid = ty * kTX + tx;
    const int x0 = blockIdx.x * kTX, y0 = blockIdx.y * kTY;
    const size_t n = (size_t)g.nr * g.nz;
    // ---- the tile and its halo: conserved state, p, v_r, v_z
    for (int idx = tid; idx < kSX * kSY; idx += kTX * kTY) {
        const int lx = idx % kSX, ly = idx / kSX;
        bool fr, fz;
        const int si = ghost_src(x0 + lx - kHalo, g.nr, g.bc[0], g.bc[1], fr);
        const int sj = ghost_src(y0 + ly - kHalo, g.nz, g.bc[2], g.bc[3], fz);
        const size_t k = (size_t)sj * g.nr + si;
        const double u0 = P.U[k], u3 = P.U[3 * n + k];
        double u1 = P.U[n + k], u2 = P.U[2 * n + k];
        if (fr) u1 = -u1;
        if (fz) u2 = -u2;
        s.u[0][ly][lx] = u0; s.u[1][ly][lx] = u1; s.u[2][ly][lx] = u2; s.u[3][ly][lx] = u3;
        s.p[ly][lx] = pressure_of(g.gamma, u0, u1, u2, u3);
        s.vr[ly][lx] = u1 / u0;
        s.vz[ly][lx] = u2 / u0;
    }
    __syncthreads();
    const double ar = P.alpha[0], az = P.alpha[1];
    const int lx = tx + kHalo, ly = ty + kHalo;
    // ---- r direction: east face by this thread, west face from the lane to the left (lane 0 recomputes it)
    double fe[4], fw[4];
    face_flux<0>(s, ly, lx, ar, fe);
#pragma unroll
    for (int c = 0; c < 4; ++c) fw[c] = __shfl_up_sync(0xffffffffu, fe[c], 1);
    if (tx == 0) face_flux<0>(s, ly, lx - 1, ar, fw);
    // ---- z direction: north face by this thread, south face from the thread row below (row 0 recomputes it)
    double gn[4], gs[4];
    face_flux<1>(s, ly, lx, az, gn);
#pragma unroll
    for (int c = 0; c < 4; ++c) s.gn[c][ty][tx] = gn[c];
    __syncthreads();
    if (ty == 0) face_flux<1>(s, ly - 1, lx, az, gs);
    else {
#pragma unroll
        for (int c = 0; c < 4; ++c) gs[c] = s.gn[c][ty - 1][tx];
    }
    const int gi = x0 + tx, gj = y0 + ty;
    if (gi >= g.nr || gj >= g.nz) return;
    const size_t k = (size_t)gj * g.nr + gi;
    double dt = 0.0;
    if (MODE != 0) dt = *P.dt;
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        const double L = -((fe[c] - fw[c]) / g.dr) - ((gn[c] - gs[c]) / g.dz);          // W6
        if (MODE == 0) P.out[c * n + k] = L;
        else {
            const double us = s.u[c][ly][lx] + dt * L;                                 // W8
            P.out[c * n + k] = MODE == 1 ? us : P.ca * P.U0[c * n + k] + P.cb * us;
        }
    }
}

}  // namespace

struct sn_weno {
    WenoGeom g;
    int device = 0, num_sms = 0;
    double* d_stage[2] = {nullptr, nullptr};      // U1, U2
    double* d_scal = nullptr;                     // [0..5] alpha of the three stages, [6] dt, [7] user alpha pair start
    double *d_io_u = nullptr, *d_io_l = nullptr;  // host entry point staging
    cudaEvent_t ev[3] = {nullptr, nullptr, nullptr};
    double st_rhs_ms = 0, st_total_ms = 0, st_launches = 0;
};

namespace {

int launch_speeds(sn_weno* h, const double* U, double* d_alpha, cudaStream_t st) {
    const size_t n = (size_t)h->g.nr * h->g.nz;
    const int blocks = (int)std::min<size_t>((n + 255) / 256, (size_t)h->num_sms * 8);
    k_weno_speeds<<<blocks, 256, 0, st>>>(h->g, U, reinterpret_cast<unsigned long long*>(d_alpha));
    WN_TRY(cudaGetLastError());
    h->st_launches += 1;
    return 0;
}

int launch_rhs(sn_weno* h, int mode, const double* U, const double* U0, double* out, const double* d_alpha,
               const double* d_dt, double ca, double cb, cudaStream_t st) {
    RhsParams P;
    P.g = h->g; P.U = U; P.U0 = U0; P.out = out; P.alpha = d_alpha; P.dt = d_dt; P.ca = ca; P.cb = cb;
    const dim3 grid((h->g.nr + kTX - 1) / kTX, (h->g.nz + kTY - 1) / kTY), block(kTX, kTY);
    if (mode == 0) k_weno_rhs<0><<<grid, block, 0, st>>>(P);
    else if (mode == 1) k_weno_rhs<1><<<grid, block, 0, st>>>(P);
    else k_weno_rhs<2><<<grid, block, 0, st>>>(P);
    WN_TRY(cudaGetLastError());
    h->st_launches += 1;
    return 0;
}

// one SSP-RK3 step, everything enqueued on st; the step ends up in d_scal[6].  march = true (sn_weno_evolve): the step
// is clamped to t_end on the device and the time in d_scal[8] / the last-step flag in d_scal[9] are advanced.
int enqueue_step(sn_weno* h, double* U, double cfl, cudaStream_t st, bool march = false, double t_end = 0.0) {
    double* a = h->d_scal;
    WN_TRY(cudaMemsetAsync(a, 0, 6 * sizeof(double), st));
    if (int rc = launch_speeds(h, U, a, st)) return rc;
    if (march) k_weno_dt_evolve<<<1, 32, 0, st>>>(h->g, a, cfl, t_end, a + 6, a + 8);
    else k_weno_dt<<<1, 32, 0, st>>>(h->g, a, cfl, a + 6);
    WN_TRY(cudaGetLastError());
    h->st_launches += 1;
    if (int rc = launch_rhs(h, 1, U, nullptr, h->d_stage[0], a, a + 6, 0.0, 1.0, st)) return rc;
    if (int rc = launch_speeds(h, h->d_stage[0], a + 2, st)) return rc;
    if (int rc = launch_rhs(h, 2, h->d_stage[0], U, h->d_stage[1], a + 2, a + 6, 0.75, 0.25, st)) return rc;
    if (int rc = launch_speeds(h, h->d_stage[1], a + 4, st)) return rc;
    // the last stage reads U (as U0) only at the cell it writes: in place
    return launch_rhs(h, 2, h->d_stage[1], U, U, a + 4, a + 6, 1.0 / 3.0, 2.0 / 3.0, st);
}

bool bad_handle(sn_weno* h) {
    if (!h) { wn_err("NULL handle"); return true; }
    return false;
}

}  // namespace

extern "C" {

const char* sn_weno_last_error(void) { return g_wn_err.c_str(); }

sn_weno* sn_weno_create(int nr, int nz, double dr, double dz, double gamma, const int* bc) {
    g_wn_err.clear();
    if (nr < 1 || nz < 1 || !(dr > 0.0) || !(dz > 0.0) || !(gamma > 1.0) || !bc || !std::isfinite(dr) ||
        !std::isfinite(gamma)) {
        wn_err("bad argument: need nr, nz >= 1, dr, dz > 0, gamma > 1, bc != NULL");
        return nullptr;
    }
    for (int k = 0; k < 4; ++k) {
        if (bc[k] < 0 || bc[k] > 2) { wn_err("bc[%d] must be 0 (outflow), 1 (reflecting) or 2 (periodic)", k); return nullptr; }
        if (bc[k] != 0 && (k < 2 ? nr : nz) < 3) { wn_err("a reflecting / periodic axis needs >= 3 cells"); return nullptr; }
    }
    if ((bc[0] == 2) != (bc[1] == 2) || (bc[2] == 2) != (bc[3] == 2)) { wn_err("periodic boundaries come in pairs"); return nullptr; }
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess || prop.major != 10) {
        cudaGetLastError();
        wn_err("no sm_100 device (this library has no CPU fallback)");
        return nullptr;
    }
    sn_weno* h = new sn_weno();
    h->g = {nr, nz, dr, dz, gamma, {bc[0], bc[1], bc[2], bc[3]}};
    h->device = dev;
    h->num_sms = prop.multiProcessorCount;
    const size_t n4 = (size_t)4 * nr * nz;
    bool ok = cudaMalloc((void**)&h->d_stage[0], n4 * sizeof(double)) == cudaSuccess &&
              cudaMalloc((void**)&h->d_stage[1], n4 * sizeof(double)) == cudaSuccess &&
              cudaMalloc((void**)&h->d_scal, 16 * sizeof(double)) == cudaSuccess;
    for (auto& e : h->ev) ok = ok && cudaEventCreate(&e) == cudaSuccess;
    if (!ok) {
        wn_err("allocation failed: %s", cudaGetErrorString(cudaGetLastError()));
        sn_weno_destroy(h);
        return nullptr;
    }
    return h;
}

void sn_weno_destroy(sn_weno* h) {
    if (!h) return;
    cudaFree(h->d_stage[0]); cudaFree(h->d_stage[1]); cudaFree(h->d_scal); cudaFree(h->d_io_u); cudaFree(h->d_io_l);
    for (auto& e : h->ev) if (e) cudaEventDestroy(e);
    delete h;
}

int sn_weno_max_speeds(sn_weno* h, const double* U, double* alpha_host, void* stream) {
    g_wn_err.clear();
    if (bad_handle(h)) return -1;
    if (!U || !alpha_host) { wn_err("NULL argument"); return -1; }
    cudaStream_t st = (cudaStream_t)stream;
    WN_TRY(cudaSetDevice(h->device));
    h->st_launches = 0;
    WN_TRY(cudaMemsetAsync(h->d_scal, 0, 2 * sizeof(double), st));
    if (int rc = launch_speeds(h, U, h->d_scal, st)) return rc;
    WN_TRY(cudaMemcpyAsync(alpha_host, h->d_scal, 2 * sizeof(double), cudaMemcpyDeviceToHost, st));
    WN_TRY(cudaStreamSynchronize(st));
    return 0;
}

int sn_weno_rhs(sn_weno* h, const double* U, double* L, double alpha_r, double alpha_z, void* stream) {
    g_wn_err.clear();
    if (bad_handle(h)) return -1;
    if (!U || !L || U == L) { wn_err("U and L must be distinct non-NULL device pointers"); return -1; }
    cudaStream_t st = (cudaStream_t)stream;
    WN_TRY(cudaSetDevice(h->device));
    h->st_launches = 0;
    WN_TRY(cudaEventRecord(h->ev[0], st));
    if (alpha_r < 0.0 || alpha_z < 0.0) {
        WN_TRY(cudaMemsetAsync(h->d_scal, 0, 2 * sizeof(double), st));
        if (int rc = launch_speeds(h, U, h->d_scal, st)) return rc;
    } else {
        const double a[2] = {alpha_r, alpha_z};
        WN_TRY(cudaMemcpyAsync(h->d_scal, a, sizeof a, cudaMemcpyHostToDevice, st));   // pageable: staged before return
    }
    WN_TRY(cudaEventRecord(h->ev[1], st));
    if (int rc = launch_rhs(h, 0, U, nullptr, L, h->d_scal, nullptr, 0.0, 0.0, st)) return rc;
    WN_TRY(cudaEventRecord(h->ev[2], st));
    return 0;
}

int sn_weno_step(sn_weno* h, double* U, double cfl, double* dt_host, void* stream) {
    g_wn_err.clear();
    if (bad_handle(h)) return -1;
    if (!U || !(cfl > 0.0)) { wn_err("bad argument: U != NULL, cfl > 0"); return -1; }
    cudaStream_t st = (cudaStream_t)stream;
    WN_TRY(cudaSetDevice(h->device));
    h->st_launches = 0;
    WN_TRY(cudaEventRecord(h->ev[0], st));
    WN_TRY(cudaEventRecord(h->ev[1], st));         // a step's three reconstructions are not timed apart: rhs_ms = total_ms
    if (int rc = enqueue_step(h, U, cfl, st)) return rc;
    WN_TRY(cudaEventRecord(h->ev[2], st));
    if (dt_host) {
        WN_TRY(cudaMemcpyAsync(dt_host, h->d_scal + 6, sizeof(double), cudaMemcpyDeviceToHost, st));
        WN_TRY(cudaStreamSynchronize(st));
    }
    return 0;
}

int sn_weno_evolve(sn_weno* h, double* U, double cfl, double t_end, int max_steps, void* stream) {
    g_wn_err.clear();
    if (bad_handle(h)) return -1;
    if (!U || !(cfl > 0.0) || !(t_end >= 0.0) || max_steps < 0) { wn_err("bad argument"); return -1; }
    cudaStream_t st = (cudaStream_t)stream;
    WN_TRY(cudaSetDevice(h->device));
    double t = 0.0;
    int steps = 0;
    double launches = 0;
    // t and the last-step flag live on the device (d_scal[8], [9]); the step, clamped to t_end, is formed there from the
    // maxima the first stage needs anyway.  One read-back per step (dt, t, flag) decides whether to go on.
    const double zero[2] = {0.0, 0.0};
    WN_TRY(cudaMemcpyAsync(h->d_scal + 8, zero, sizeof zero, cudaMemcpyHostToDevice, st));    // pageable: staged before return
    while (t < t_end && steps < max_steps) {
        h->st_launches = 0;
        if (int rc = enqueue_step(h, U, cfl, st, true, t_end)) return rc;
        launches += h->st_launches;
        double back[4] = {0.0, 0.0, 0.0, 0.0};                       // d_scal[6..9] = dt, (unused), t, last-step flag
        WN_TRY(cudaMemcpyAsync(back, h->d_scal + 6, sizeof back, cudaMemcpyDeviceToHost, st));
        WN_TRY(cudaStreamSynchronize(st));
        if (!(back[0] > 0.0)) { wn_err("non-positive or non-finite time step at step %d", steps); return -2; }
        t = back[2];
        ++steps;
        if (back[3] != 0.0) break;
    }
    h->st_launches = launches;
    return steps;
}

int sn_weno_rhs_host(sn_weno* h, const double* U_host, double* L_host, void* stream) {
    g_wn_err.clear();
    if (bad_handle(h)) return -1;
    if (!U_host || !L_host) { wn_err("NULL argument"); return -1; }
    cudaStream_t st = (cudaStream_t)stream;
    WN_TRY(cudaSetDevice(h->device));
    const size_t bytes = (size_t)4 * h->g.nr * h->g.nz * sizeof(double);
    if (!h->d_io_u) {
        WN_TRY(cudaMalloc((void**)&h->d_io_u, bytes));
        WN_TRY(cudaMalloc((void**)&h->d_io_l, bytes));
    }
    WN_TRY(cudaMemcpyAsync(h->d_io_u, U_host, bytes, cudaMemcpyHostToDevice, st));
    if (int rc = sn_weno_rhs(h, h->d_io_u, h->d_io_l, -1.0, -1.0, stream)) return rc;
    WN_TRY(cudaMemcpyAsync(L_host, h->d_io_l, bytes, cudaMemcpyDeviceToHost, st));
    WN_TRY(cudaStreamSynchronize(st));
    return 0;
}

int sn_weno_get_stat(sn_weno* h, const char* key, double* out) {
    g_wn_err.clear();
    if (!h || !key || !out) { wn_err("NULL argument"); return -1; }
    if (!strcmp(key, "launches")) { *out = h->st_launches; return 0; }
    if (!strcmp(key, "rhs_ms") || !strcmp(key, "total_ms")) {
        // the events of the last rhs / step call: [0] start, [1] before the (last) rhs kernel, [2] end
        if (cudaEventSynchronize(h->ev[2]) != cudaSuccess) { cudaGetLastError(); wn_err("no timed call yet"); return -1; }
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, !strcmp(key, "rhs_ms") ? h->ev[1] : h->ev[0], h->ev[2]) != cudaSuccess) {
            cudaGetLastError();
            wn_err("no timed call yet");
            return -1;
        }
        *out = ms;
        return 0;
    }
    wn_err("unknown stat '%s'", key);
    return -1;
}

}  // extern "C"
