// common.cuh -- shared device-side types of the sn_poisson library (sm_100a only).
// Discretisation and pinned arithmetic: DESIGN.md §2-3; PAPER.md:91,99 for the physics.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace snp {

constexpr double kFourPi = 12.566370614359172;   // 4*pi rounded to fp64 (R10)
constexpr double kPi = 3.141592653589793;
constexpr int kMaxL = 64;

// Per-member control block.  Result fields are written by the device-side stopping decision (step a-3); the
// "director" fields drive the blocked path (sweep_blocked.cuh), where the last CTA of every launch decides what
// the next launch does for this member.
struct Ctl {
    int done;          // 1 once the member is finished (result fields valid, phi_inout holds the result)
    int sweeps;        // full sweeps applied to the returned phi
    int status;        // 0 / 1 / -3 as in sn_poisson_result
    int panic;         // resident path watchdog: non-zero = a wait exceeded its budget (code of the first one)
    double residual;   // R_k of the last applied sweep
    double maxf;       // max |4 pi rho| (written by the moments pass)
    // ---- director state (blocked path) ----
    int action;        // what the next launch does: kActSkip / kActAdvance / kActRedo / kActReplay / kActCopy
    int src;           // buffer the action reads (0 = caller's phi_inout, 1 = workspace); it writes the other one
    int k0;            // sweeps already applied in the state it reads
    int n;             // sweeps it runs
    int track;         // TrackMode of the run
    int fin_sweeps;    // result to publish once a replay / copy has completed
    int fin_status;
    unsigned int arrived;   // CTAs of this member that have finished the current launch
    double fin_R;
    int panic_tile, panic_arg;   // where the watchdog tripped (diagnostics)
};

enum BlockedAction : int { kActSkip = 0, kActAdvance = 1, kActRedo = 2, kActReplay = 3, kActCopy = 4 };

// Grid geometry + coefficient tables; passed by value to every kernel.
struct Geom {
    int nr, nz, symmetry, lmax;
    double dr, dz;
    double iz2;        // 1/dz^2
    double D, D0;      // 2/dr^2+2/dz^2 and D - 1/dz^2 (reflecting-equator row)
    double wD, wD0;    // omega/D, omega/D0
    double tol;
    const double* cE;  // [nr]  ((i+1)/(i+1/2))/dr^2
    const double* cW;  // [nr]  (i/(i+1/2))/dr^2, cW[0] = 0: regular axis
    // stopping rule (R9 / R16): 0 = residual ratio R_k, 1 = the paper-literal relative change E_k.  Rule 1 with
    // symmetry = 1 also needs the maximum of |res| over the reflecting-equator row alone (its omega/diag differs):
    int rule;
    int slots0_stride;                  // per member
    unsigned int* slots0_f;             // [nb][cap]  upper words (FAST)
    unsigned long long* slots0_x;       // [nb][cap]  exact keys
};

__device__ __forceinline__ unsigned long long dbits(double x) { return (unsigned long long)__double_as_longlong(x); }
__device__ __forceinline__ double bits2d(unsigned long long b) { return __longlong_as_double((long long)b); }

// |x| as an order-preserving unsigned key (non-negative doubles order like their bit patterns; NaN sorts highest,
// so a NaN anywhere is sticky in a max-reduction, like the oracle's).
__device__ __forceinline__ unsigned long long abs_key(double x) { return dbits(x) & 0x7fffffffffffffffull; }

__device__ __forceinline__ unsigned long long warp_max_u64(unsigned long long v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        unsigned long long t = __shfl_xor_sync(0xffffffffu, v, o);
        v = t > v ? t : v;
    }
    return v;
}

// Stopping ratio of one sweep (R9): R = Rabs / fma(D, P, maxf); Rabs == 0 -> 0.
__device__ __forceinline__ double stop_ratio(unsigned long long rabs_key, unsigned long long p_key, double maxf,
                                             double D) {
    const double Rabs = bits2d(rabs_key);
    if (Rabs == 0.0) return 0.0;
    return __ddiv_rn(Rabs, __fma_rn(D, bits2d(p_key), maxf));
}

// The value the stopping rule compares with tol after a sweep (keys: max|res|, max|phi_new| over all cells, max|res|
// over the reflecting-equator row).  Rule 0: R_k (above).  Rule 1 (R16; "relative changes of all
// grids"): E_k = max|dphi| / max|phi_new| with dphi = w_j (x) res.  Rounded multiplication by a positive constant is
// monotone, so max_j |w_j (x) res| = max(wD (x) max|res|, wD0 (x) max_row0|res|) EXACTLY (wD0 > wD makes the row-0 cells
// inside the first maximum harmless); max|dphi| == 0 -> 0.
__device__ __forceinline__ double stop_value(const Geom& g, unsigned long long rabs_key, unsigned long long p_key,
                                             unsigned long long r0_key, double maxf) {
    if (g.rule == 0) return stop_ratio(rabs_key, p_key, maxf, g.D);
    unsigned long long c = abs_key(__dmul_rn(g.wD, bits2d(rabs_key)));
    if (g.symmetry == 1) {
        const unsigned long long c0 = abs_key(__dmul_rn(g.wD0, bits2d(r0_key)));
        c = c0 > c ? c0 : c;                         // keys: NaN sorts highest (sticky)
    }
    if (c == 0ull) return 0.0;
    return __ddiv_rn(bits2d(c), bits2d(p_key));
}

__device__ __forceinline__ bool is_nonfinite(double x) { return !(x == x) || x == INFINITY || x == -INFINITY; }

// One SOR cell update with the pinned expression tree (R10).  Returns the new value; res_out = pre-update
// residual f - L(phi).
__device__ __forceinline__ double sor_update(double cE, double cW, double cN, double cS, double diag, double w,
                                             double pE, double pW, double pN, double pS, double pC, double f,
                                             double& res_out) {
    double t = __dmul_rn(cE, pE);
    t = __fma_rn(cW, pW, t);
    t = __fma_rn(cN, pN, t);
    t = __fma_rn(cS, pS, t);
    t = __fma_rn(-diag, pC, t);
    const double res = __dsub_rn(f, t);
    res_out = res;
    return __fma_rn(-w, res, pC);
}

}  // namespace snp
