// xy_device.cuh -- device-side building blocks of the XY Swendsen-Wang sweep for sm_100a:
// Philox4x32-10, the filtered bond decision, the reflection, global union-find helpers,
// warp / block reductions.  Product code: shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace xy {

// Programmatic dependent launch (sm_90+; cudaLaunchAttributeProgrammaticStreamSerialization): the kernels of a sweep
// are launched so that the NEXT kernel of the stream may become resident while this grid drains and run its prologue
// (whatever touches no data of its predecessor).  pdl_wait() returns once the preceding grid has completed and its
// writes are visible; pdl_launch_next() allows the next grid to be scheduled.  Every kernel calls them in this order,
// wait first: a grid that could be scheduled before its predecessor passed its own wait could read (in its prologue)
// data that a kernel two steps back is still writing.  Both are no-ops in a launch without the attribute.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_next() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

constexpr double kTwoPi = 6.283185307179586;   // fl64(2 pi)
constexpr double kPi    = 3.141592653589793;   // fl64(pi)

// Checked build (-DXY_CHECKED, see profiles/r2_checked_build.md): every index the kernels derive from data
// (table entry, tile-local parent offset, queue slot, label chased in global memory) is range-checked and
// violations are counted per site of the check; the normal build compiles the checks away.  This stands in
// for compute-sanitizer memcheck, which is closed on the pool this was developed on.
#ifdef XY_CHECKED
__device__ unsigned long long g_xy_check_fail[8];
#define XY_CHECK(code, cond) do { if (!(cond)) atomicAdd(&xy::g_xy_check_fail[code], 1ULL); } while (0)
#else
#define XY_CHECK(code, cond) do { } while (0)
#endif
enum : int { CHK_TABLE = 0, CHK_PARENT = 1, CHK_WLIST = 2, CHK_GLABEL = 3, CHK_QUEUE = 4, CHK_LOC = 5 };

enum : uint32_t { TAG_INIT = 0, TAG_DIR = 1, TAG_BOND = 2, TAG_FLIP = 3, TAG_BOND_LO = 4 };

// ---------------------------------------------------------------------------------------------
// Philox4x32 with 10 rounds (Salmon et al., SC'11).  Counter (c0..c3), key (k0,k1).
// IMAD.WIDE.U32 gives hi and lo of each product in one instruction.
// ---------------------------------------------------------------------------------------------
struct U4 { uint32_t x, y, z, w; };

__host__ __device__ __forceinline__ U4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                                      uint32_t k0, uint32_t k1)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        const uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    return U4{c0, c1, c2, c3};
}

// The same with the ten round keys precomputed (rk[2r] = k0 + r * 0x9E3779B9, rk[2r+1] = k1 + r * 0xBB67AE85):
// as kernel arguments they are constant-bank operands of the XORs.
__device__ __forceinline__ U4 philox4x32_10_rk(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, const uint32_t (&rk)[20])
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        const uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ rk[2 * r];
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ rk[2 * r + 1];
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
    }
    return U4{c0, c1, c2, c3};
}

// counter = (idx lo, idx hi, (u32)t, tag); key = (seed lo, seed hi)
__host__ __device__ __forceinline__ U4 rng(uint32_t seed_lo, uint32_t seed_hi, uint64_t idx, uint32_t t, uint32_t tag)
{
    return philox4x32_10((uint32_t)idx, (uint32_t)(idx >> 32), t, tag, seed_lo, seed_hi);
}

// ---------------------------------------------------------------------------------------------
// Bond decision.  Definition (fp64): active iff u < p, u = (w + 0.5) 2^-32,
// p = -expm1(-2 beta sigma_i sigma_j), sigma = cos(theta - phi).
// ---------------------------------------------------------------------------------------------
__device__ __noinline__ bool bond_exact(float ti, float tj, double phi, double beta, uint32_t w,
                                        unsigned long long *fallback_counter)
{
    const double si = cos(__dsub_rn((double)ti, phi));
    const double sj = cos(__dsub_rn((double)tj, phi));
    const double a = __dmul_rn(si, sj);
    const double x = __dmul_rn(__dmul_rn(-2.0, beta), a);
    const double p = -expm1(x);
    const double u = __dmul_rn(__dadd_rn((double)w, 0.5), 1.0 / 4294967296.0);
    atomicAdd(fallback_counter, 1ULL);
    return u < p;
}

// The same for the bond of site (y, x) in direction dir (0: +x, 1: +y), angles re-read from memory
// (the streaming loop does not keep them once (cos, sin, sigma) are evaluated).
// wrap_rows: number of rows after which y wraps to row 0 (0: never: a slab, whose row below the last is its halo row)
__device__ __noinline__ bool bond_exact_at(const float *theta, uint32_t L, uint32_t wrap_rows, uint32_t y, uint32_t x, int dir,
                                           double phi, double beta, uint32_t w, unsigned long long *fallback_counter)
{
    uint32_t x2 = x, y2 = y;
    if (dir == 0) { x2 = x + 1; if (x2 == L) x2 = 0; }
    else { y2 = y + 1; if (y2 == wrap_rows) y2 = 0; }
    return bond_exact(theta[(size_t)y * L + x], theta[(size_t)y2 * L + x2], phi, beta, w, fallback_counter);
}

// Filter (fp32, on the 16 leading bits of u): e32 = ex2.approx((sigma_i m2b) sigma_j), m2b = -2 beta
// log2(e), approximates e = 1 - p = exp(-2 beta sigma_i sigma_j); f = 1 + v with
// v = ((65535 - h) + 0.5) 2^-16 the midpoint of the interval that 1 - u lies in when only the leading
// 16 bits h of the random word are known, so d = (e32 + 1) - f approximates e - (1 - u), and
//     u < p  <=>  e < 1 - u  <=>  d < 0.
// Error budget of d (sigma from k_bonds' fp32 table path, |delta sigma| <= 1e-7 ABSOLUTE: two table
// roundings and two fused roundings of 2^-25 each, truncation 2e-11):
//   exponent y = (sigma_i m2b) sigma_j: three fp32 roundings (m2b, two products), relative 1.8e-7,
//     -> |delta e| <= e ln2 |y| 1.8e-7 <= 0.531 * 0.693 * 1.8e-7 = 6.6e-8 (y 2^-y <= 0.531 for y <= 0;
//     for y > 0 the true e exceeds 1 and no error of this size can bring e32 below 1 - delta);
//   the absolute sigma errors: |delta y| <= |m2b| (|sigma_i| + |sigma_j|) 1e-7, so
//     |delta e| <= 2 beta (|sigma_i| + |sigma_j|) exp(-2 beta sigma_i sigma_j) 1e-7 <= 4e-7 beta;
//   ex2.approx: 2^-22 relative <= 2.4e-7;  e32 + 1: 6e-8;  f subtracts exactly;
//   the unknown trailing bits of u: 2^-17 = 7.63e-6.
// Total < 8.0e-6 + 4e-7 beta.  |d| > delta(beta) = 1.2e-5 + 1e-6 beta (margin >= 1.4 at every beta)
// settles the sign; otherwise (2 delta of all bonds: 2.6e-5 at beta = 1.12) the trailing bits are
// drawn and the definition is evaluated in fp64 (bond_exact).  At huge beta delta exceeds every |d|
// and all decisions take the exact path.
__host__ __device__ __forceinline__ float filter_delta(double beta)
{
    return (float)(1.2e-5 + 1.0e-6 * beta);
}

struct BondCtx {
    double phi, beta;
    float m2b;                                  // -2 beta log2(e), fp32
    float delta;                                // filter_delta(beta)
    unsigned long long *fallback_counter;
};

// gs = sigma_i * m2b (fp32), gj = sigma_j (fp32); hs holds the 16 leading bits h of the random word
// at bit positions 7..22 (other bits arbitrary); returns d (see above)
__device__ __forceinline__ float bond_filter(float gs, float gj, uint32_t hs)
{
    float e;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e) : "f"(gs * gj));
    const float f = __uint_as_float(((~hs) & 0x007fff80u) | 0x3f800040u);
    return (e + 1.0f) - f;
}

// ---------------------------------------------------------------------------------------------
// Reflection theta -> 2 phi + pi - theta (mod 2pi), specified to the rounding: A is computed once
// per sweep on the host (A = 2 phi + pi reduced into [0, 2pi)); here only add/sub/convert.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ float reflect(float theta, double A)
{
    double d = __dsub_rn(A, (double)theta);
    // "while (d < 0) d += 2pi": A >= 0 and theta <= fl32(2pi) < 2 * 2pi64 give d > -2 * 2pi64, so twice is enough
    // the sign is read from the high word (integer compare instead of an fp64 one; A - theta is never -0.0)
    if (__double2hiint(d) < 0) d = __dadd_rn(d, kTwoPi);
    if (__double2hiint(d) < 0) d = __dadd_rn(d, kTwoPi);
    return __double2float_rn(d);
}

// ---------------------------------------------------------------------------------------------
// Union-find in global memory (boundary merge; the tile-local one lives with k_label).  Links always
// go from the larger to the smaller index, so the root of a component is its minimum index.
// ---------------------------------------------------------------------------------------------
template <typename T> struct AtomT;
template <> struct AtomT<uint32_t> { using type = unsigned int; };
template <> struct AtomT<uint64_t> { using type = unsigned long long; };

template <typename LabelT>
__device__ __forceinline__ LabelT gload(const LabelT *p)        // L2-coherent load (other SMs update concurrently)
{
    return __ldcg(p);
}

template <typename LabelT>
__device__ __forceinline__ LabelT gfind(LabelT *lab, LabelT a)
{
    LabelT r = gload(lab + a);
    while (r != a) { XY_CHECK(CHK_GLABEL, r < a); a = r; r = gload(lab + a); }
    return a;
}

// find with path halving; the re-pointing is an atomicMin (parents only ever decrease: ancestors
// have smaller indices), so it can never undo a concurrent min-link of the same entry.
template <typename LabelT>
__device__ __forceinline__ LabelT gfind_h(LabelT *lab, LabelT a)
{
    using A = typename AtomT<LabelT>::type;
    LabelT r = gload(lab + a);
    while (r != a) {
        const LabelT g = gload(lab + r);
        if (g == r) return r;
        atomicMin(reinterpret_cast<A *>(lab + a), (A)g);
        a = g;
        r = gload(lab + a);
    }
    return a;
}

// a and b are most likely still roots (labels straight from k_label): try the link before any find.
// atomicMin on lab[hi] with lo < hi is a valid step whatever hi is: if hi was a root (old == hi) it
// is now linked into lo's component; if not, hi hangs under min(old, lo) and old, lo remain to be united.
template <typename LabelT>
__device__ __forceinline__ void gunion(LabelT *lab, LabelT a, LabelT b)
{
    using A = typename AtomT<LabelT>::type;
    if (a == b) return;
    {
        const LabelT hi = a > b ? a : b, lo = a > b ? b : a;
        const LabelT old = (LabelT)atomicMin(reinterpret_cast<A *>(lab + hi), (A)lo);
        if (old == hi || old == lo) return;
        a = old;
        b = lo;
    }
    for (;;) {
        a = gfind_h(lab, a);
        b = gfind_h(lab, b);
        if (a == b) return;
        if (a < b) { const LabelT t = a; a = b; b = t; }
        const LabelT old = (LabelT)atomicMin(reinterpret_cast<A *>(lab + a), (A)b);
        if (old == a) return;
        a = old;
    }
}

// ---------------------------------------------------------------------------------------------
// Reductions with a fixed summation tree (bitwise reproducible for a fixed launch shape).
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

__device__ __forceinline__ unsigned long long warp_sum_u64(unsigned long long v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

}  // namespace xy
