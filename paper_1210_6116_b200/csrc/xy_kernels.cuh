// xy_kernels.cuh -- the kernels of one Swendsen-Wang sweep of the 2D XY model on sm_100a.
//
//   k_bonds   (S2, and S7 of the incoming configuration): warps stream strips of the lattice row
//             by row: theta is split exactly on a 2^-10 grid in fp32; sigma (fp32) and (cos, sin)
//             (fp64) per site come from two shared-memory tables and a second-order rotation ->
//             observables, Philox bond draws, filtered bond decisions -> packed bond bits
//             (0.25 B/site).  theta is read once (+ halo); no block barrier in the loop.
//   k_label   (S3): one CTA per TW x TH tile, integer only, bit-parallel: a thread holds the x / y
//             bond bits of 32 sites in two registers; union-find over RUNS of x bonds in shared
//             memory, united in log2(TH) waves -> provisional label (global index of the
//             tile-local root) and one root bit per site, written once.
//   k_merge   (S4): one thread per tile-edge bond; atomicMin union-find on the label array.
//   k_flip    (S5+S6): coins of a tile's labels from one Philox call per tile row; tile roots
//             that k_merge linked elsewhere chase their root; reflect, write theta back.
//   finalize       (S8): the last CTA of k_bonds reduces the per-CTA partial sums in a fixed
//                  order, writes the per-sweep record and advances the PCC controller.
//
// Layouts: theta fp32 row-major i = y*L + x.  labels LabelT (u32 or u64) same indexing.
// bonds packed 2 bits/site: byte (i>>2) holds bx(4k+j) in bit j and by(4k+j) in bit 4+j.
#pragma once
#include "xy_device.cuh"
#include "../../include/xy.h"

namespace xy {

constexpr int kPartialStride = 16;         // doubles per CTA partial record: 14 sums + 2 counts

// Device-resident control block: PCC controller (O8) + counters.
struct DevCtl {
    double   beta;                // beta of the next sweep when PCC runs on the device
    double   dbeta;
    double   acc_e, acc_s2;
    unsigned long long k;         // measured sweeps fed so far
    unsigned long long n_dec;
    double   stage_sum, last_sum;
    unsigned long long stage_cnt, last_cnt;
    // schedule
    unsigned long long halve_every;
    double   dbeta_min, target;
    unsigned int window, dirs;
    // trace
    double  *trace_beta, *trace_bY;
    unsigned long long trace_cap;
    unsigned long long trace_base;   // decisions taken before this call: entry n_dec - trace_base of the trace arrays
    // misc
    unsigned long long fallback_count;
    unsigned int ticket;          // last-block-done counter of k_bonds
    unsigned int pad;
    // sums over the measured sweeps fed to the controller (xy_pcc_state): <m^2> and chi(k) of a long run without
    // reading the per-sweep ring back
    double   sum_m2, sum_chik;
    unsigned long long n_acc;
    // slab: edge sites of the gathered record that name a root outside this slab (wrong rank / order of the gather);
    // k_stitch_apply skips them and counts them here, the next blocking call of the slab reports XY_ERR_ARG
    unsigned int stitch_bad;
    unsigned int pad2;
};

struct SweepArgs {
    float       *theta;
    void        *labels;
    uint8_t     *bonds;
    uint32_t    *rootmask;        // 1 bit per site: the site is the root of its tile-local component (k_label -> k_flip)
    double      *partials;        // [grid][kPartialStride]
    DevCtl      *ctl;
    xy_obs      *ring;
    uint32_t     ring_cap;
    uint32_t     L;
    uint32_t     tiles_x, ntiles;
    uint32_t     Ldiv_mul, Ldiv_shift;   // d / L for d < 2^22: umulhi(d, Ldiv_mul) >> Ldiv_shift
    uint32_t     seed_lo, seed_hi;
    uint32_t     rk[20];          // Philox round keys (k0, k1) of rounds 0..9, derived from the seed on the host
    uint32_t     t;               // sweep counter of THIS sweep (state before it has T = t sweeps done)
    int          beta_from_ctl;   // 1: read beta from ctl->beta (PCC), 0: use beta
    int          feed_pcc;        // 1: finalize feeds the observables of the incoming state to the controller
    int          obs_fill;        // 1: finalize writes the observables of the incoming state into ring[T]
    double       beta;
    double       phi, cphi, sphi, A;
    const double2 *sincos_tab;    // [kTabN + 1] (cos, sin)(k / 1024), host-computed
    double       ck1, sk1;        // (cos, sin)(2 pi / L)
    xy_fourier  *fring;           // ring of structure-factor records (XY_FLAG_FOURIER), else NULL
    // slab of a lattice sharded by rows: the state holds rows [y_off, y_off + rows) of the
    // L x L lattice; rows == L, y_off == 0, open_y == 0 for a whole lattice
    uint32_t     rows, y_off;
    int          open_y;          // 1: no periodic wrap in y: row `rows` of theta is the halo row (the neighbour's first
                                  //    row), the y bonds of the last row are left to the stitch
    const uint64_t *xroot;        // slab: global canonical roots of the local roots the stitch overrode (k_flip)
};

// slab mode: label[r] of a local root r whose cluster reaches into another slab and has its canonical root there is
// kSlabSpecial | k: its global root is xroot[k] (labels are u32 words in slab mode, local indices below 2^31)
constexpr uint32_t kSlabSpecial = 0x80000000u;


template <int VEC> struct FVec;
template <> struct FVec<4> { using type = float4; };
template <> struct FVec<2> { using type = float2; };

// RO: the array is read-only for the whole kernel (ld.global.nc); otherwise a plain load.
template <int VEC, bool RO>
__device__ __forceinline__ void load_vec(const float *p, float (&out)[VEC])
{
    if constexpr (VEC == 4) {
        const float4 v = RO ? __ldg(reinterpret_cast<const float4 *>(p)) : *reinterpret_cast<const float4 *>(p);
        out[0] = v.x; out[1] = v.y; out[2] = v.z; out[3] = v.w;
    } else {
        const float2 v = RO ? __ldg(reinterpret_cast<const float2 *>(p)) : *reinterpret_cast<const float2 *>(p);
        out[0] = v.x; out[1] = v.y;
    }
}

// PCC controller step, the arithmetic of DESIGN.md section 3 (O8) in this exact order.
__device__ inline void pcc_feed(DevCtl *c, double N, double Cx, double Sx, double Cy, double Sy, double Mx, double My, double chik)
{
    c->sum_m2 = __dadd_rn(c->sum_m2, __ddiv_rn(__dadd_rn(__dmul_rn(Mx, Mx), __dmul_rn(My, My)), __dmul_rn(N, N)));
    c->sum_chik = __dadd_rn(c->sum_chik, chik);
    c->n_acc += 1;
    double e, s2;
    if (c->dirs == 2) {
        e = __ddiv_rn(__dadd_rn(Cx, Cy), __dmul_rn(2.0, N));
        const double sx2 = __dmul_rn(Sx, Sx), sy2 = __dmul_rn(Sy, Sy);
        s2 = __ddiv_rn(__dadd_rn(sx2, sy2), __dmul_rn(__dmul_rn(2.0, N), N));
    } else {
        e = __ddiv_rn(Cx, N);
        const double sx = __ddiv_rn(Sx, N);
        s2 = __dmul_rn(sx, sx);
    }
    c->k += 1;
    c->acc_e = __dadd_rn(c->acc_e, e);
    c->acc_s2 = __dadd_rn(c->acc_s2, s2);
    if (c->k % c->window == 0) {
        const double w = (double)c->window;
        const double ae = __ddiv_rn(c->acc_e, w);
        const double as2 = __ddiv_rn(c->acc_s2, w);
        const double bn = __dmul_rn(c->beta, N);
        const double Y = __dsub_rn(ae, __dmul_rn(bn, as2));
        const double bY = __dmul_rn(c->beta, Y);
        if (c->trace_beta && c->n_dec - c->trace_base < c->trace_cap) {
            c->trace_beta[c->n_dec - c->trace_base] = c->beta;
            c->trace_bY[c->n_dec - c->trace_base] = bY;
        }
        c->stage_sum = __dadd_rn(c->stage_sum, c->beta);
        c->stage_cnt += 1;
        c->n_dec += 1;
        c->beta = (bY < c->target) ? __dadd_rn(c->beta, c->dbeta) : __dsub_rn(c->beta, c->dbeta);
        c->acc_e = 0.0;
        c->acc_s2 = 0.0;
    }
    if (c->halve_every && c->k % c->halve_every == 0) {
        const double h = __ddiv_rn(c->dbeta, 2.0);
        const double nd = h > c->dbeta_min ? h : c->dbeta_min;
        if (nd != c->dbeta) {
            if (c->stage_cnt > 0) { c->last_sum = c->stage_sum; c->last_cnt = c->stage_cnt; }
            c->stage_sum = 0.0;
            c->stage_cnt = 0;
        }
        c->dbeta = nd;
    }
}

// ---------------------------------------------------------------------------------------------
// k_bonds (S2, and S7 of the incoming configuration): streaming, no block barrier in the loop.
// A warp walks strips of TW = 32*VEC columns x RS rows, top to bottom, one row per iteration,
// carrying the previous row's (cos, sin, sigma) in registers; lane l owns VEC consecutive sites.
// Right neighbour of a lane's last site: shuffle from lane+1; for lane 31 the strip's halo column,
// computed once per strip by lanes 0..RS-1 into a per-warp shared slot.  Row RS of the strip (the
// first row of the strip below) is recomputed as the y-halo (1/RS overhead).
//
// Angle -> (cos, sin)(theta - phi) per site; sigma IS the cosine.  theta is split EXACTLY in fp32 on
// the grid h = k 2^-10:
//   tm = theta + 1.5 2^13 (round to nearest: ulp 2^-10), h = tm - 1.5 2^13, x = theta - h,
//   |x| <= 2^-11, all three exact; k = tm's mantissa bits above 2^22 (bits(tm) - bits(1.5 2^13)), 0 <= k <= 6434.
// The table of the sweep, (C_k, S_k) = (cos, sin)(k 2^-10 - phi), is rotated at kernel start from the
// host-computed (cos, sin)(k 2^-10) into shared memory (fp64 with observables, fp32 without), and
//   (cos, sin)(theta - phi) = (C_k w - S_k x, S_k w + C_k x), w = 1 - x^2/2:
//   one conversion of x (exact) and 6 fp64 operations, sigma = that cosine rounded to fp32; without
//   observables 4 fp32 operations on the fp32 table.  Truncation: |sin x - x| <= x^3/6 <= 1.95e-11,
//   |cos x - w| <= x^4/24 <= 2.4e-15; table entries within 3e-16.
// The link sums Cx, Sx, Cy, Sy depend on angle differences only, so they are the same in the rotated
// frame; Mx, My (and the structure-factor sums) are linear in (cos, sin) and are rotated back by phi
// once, in finalize.
// kFourier: also reduce the 8 structure-factor sums at k = 2 pi / L (x and y direction) of the
// incoming configuration (Eq. 8-9): per-column sums of (cos, sin) live in registers
// for the rows of a strip and meet e^{ik x} once per strip; per-row sums meet e^{ik y} once per row.
// kObs = false (xy_set_obs_mode(XY_OBS_NONE)): fp32 only, no fp64 table, no sums; bond counts only.
// ---------------------------------------------------------------------------------------------
constexpr int kTabN = 6434;                 // table entries k = 0..kTabN at angle k / 1024; 6434/1024 >= fl32(2 pi)
constexpr float kTabMagic = 12288.0f;       // 1.5 * 2^13: fp32 ulp 2^-10 in [2^13, 2^14)
// warps per CTA of k_bonds: with observables one CTA of 12 warps per SM (168 registers per thread, no spills: measured
// 0.78 ms against 0.82 at 16 warps x 128 registers and 0.91 at 8 or 10 warps); without, two CTAs of 8 warps x 128 registers
template <bool kObs> struct BondsShape { static constexpr int warps = kObs ? 12 : 8, min_ctas = kObs ? 1 : 2; };

template <bool kObs>
constexpr size_t k_bonds_smem_bytes()
{
    return (size_t)(kTabN + 1) * (kObs ? sizeof(double2) : sizeof(float2)) + 16;
}

// one table, indexed by byte offset: entries are double2 with observables, float2 without
template <bool kObs>
struct BondsEntry { static constexpr uint32_t bytes = kObs ? 16u : 8u; };

// tab_adj = shared-space byte address of entry 0 minus bits(kTabMagic) * entry size (mod 2^32): the entry
// of an angle is one multiply-add away from the bits of tm
template <bool kBonds, bool kObs>
__device__ __forceinline__ void site_eval(float theta, uint32_t tab_adj, float &g, double &c, double &s)
{
    const float tm = __fadd_rn(theta, kTabMagic);
    const float h = __fadd_rn(tm, -kTabMagic);
    const float x = __fadd_rn(theta, -h);
    const uint32_t addr = __float_as_uint(tm) * BondsEntry<kObs>::bytes + tab_adj;
    XY_CHECK(CHK_TABLE, __float_as_uint(tm) - __float_as_uint(kTabMagic) <= (uint32_t)kTabN);
    if constexpr (kObs) {
        double C, S;
        asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(C), "=d"(S) : "r"(addr));
        const double xd = (double)x;
        const double w = __fma_rn(xd * xd, -0.5, 1.0);
        c = __fma_rn(-S, xd, C * w);
        s = __fma_rn(C, xd, S * w);
        if constexpr (kBonds) g = __double2float_rn(c);
    } else {
        float C, S;
        asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(C), "=f"(S) : "r"(addr));
        const float dc = (-0.5f * x) * x;
        g = fmaf(-S, x, fmaf(C, dc, C));
    }
}

// Cold path of k_bonds: some decision of this lane's VEC sites in row gy was too close for the filter.
// Everything is recomputed from the values the hot loop still holds (sigma of the row, of the row below and
// of the right neighbour), so the hot loop keeps no per-bond state alive for it: call A again, call B for
// the trailing bits, the same filter arithmetic (bit-identical d), and the fp64 definition for every bond
// with |d| <= delta.  bits = xn | yn << 8 as the filter decided them; returns the corrected bits.
template <int VEC> struct RowSigma { float pg[VEC], g[VEC], gn; };

template <int VEC>
__device__ __noinline__ uint32_t bonds_fix(const float *theta, uint32_t L, uint32_t wrap_rows, uint32_t seed_lo, uint32_t seed_hi, uint32_t t,
                                           BondCtx bcx, uint64_t quad, uint32_t gy, uint32_t xl, RowSigma<VEC> rs, uint32_t bits)
{
    const U4 wA = rng(seed_lo, seed_hi, quad, t, TAG_BOND);
    const U4 wB = rng(seed_lo, seed_hi, quad, t, TAG_BOND_LO);
    uint32_t wa[VEC], wb[VEC];
    if constexpr (VEC == 4) {
        wa[0] = wA.x; wa[1] = wA.y; wa[2] = wA.z; wa[3] = wA.w;
        wb[0] = wB.x; wb[1] = wB.y; wb[2] = wB.z; wb[3] = wB.w;
    } else {
        const bool up = (xl & 2u) != 0;
        wa[0] = up ? wA.z : wA.x; wa[1] = up ? wA.w : wA.y;
        wb[0] = up ? wB.z : wB.x; wb[1] = up ? wB.w : wB.y;
    }
#pragma unroll
    for (int v = 0; v < VEC; ++v) {
        const float g2 = (v + 1 < VEC) ? rs.pg[(v + 1) % VEC] : rs.gn;
        const float gs = rs.pg[v] * bcx.m2b;
        const float dx = bond_filter(gs, g2, wa[v] << 7);
        const float dy = bond_filter(gs, rs.g[v], wa[v] >> 9);
        if (!(fabsf(dx) > bcx.delta)) {
            const uint32_t wx = (wa[v] << 16) | (wb[v] & 0xffffu);
            bits &= ~(1u << v);
            if (bond_exact_at(theta, L, wrap_rows, gy, xl + v, 0, bcx.phi, bcx.beta, wx, bcx.fallback_counter)) bits |= 1u << v;
        }
        if (!(fabsf(dy) > bcx.delta)) {
            const uint32_t wy = (wa[v] & 0xffff0000u) | (wb[v] >> 16);
            bits &= ~(0x100u << v);
            if (bond_exact_at(theta, L, wrap_rows, gy, xl + v, 1, bcx.phi, bcx.beta, wy, bcx.fallback_counter)) bits |= 0x100u << v;
        }
    }
    return bits;
}

// kSlab: the state is a slab of rows of a sharded lattice: `rows` rows, no wrap in y (row `rows`
// of theta is the halo row), quad indices (Philox counters) of the whole lattice.
template <int VEC, int RS, bool kBonds, bool kObs, bool kFourier, bool kSlab = false>
__global__ void __launch_bounds__(BondsShape<kObs>::warps * 32, BondsShape<kObs>::min_ctas)
k_bonds(const SweepArgs a)
{
    static_assert(!(kSlab && kFourier), "slabs do not reduce the structure-factor sums");
    static_assert(kObs || !kFourier, "the structure-factor sums are observables");
    static_assert(kBonds || kObs, "nothing to do");
    constexpr int NW = BondsShape<kObs>::warps;
    constexpr int NS = kFourier ? 14 : 6;      // fp64 sums per thread / warp / CTA
    constexpr int TW = 32 * VEC;
    static_assert(RS <= 32, "halo column is computed by one lane per row");

    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ double h_c[kObs ? NW : 1][RS], h_s[kObs ? NW : 1][RS];
    __shared__ float h_g[kBonds ? NW : 1][RS];
    __shared__ double red[NW][NS];
    __shared__ double2 h_ky[kFourier ? NW : 1][RS];      // (cos, sin)(2 pi y / L) of the strip's rows
    __shared__ unsigned long long redc[NW][2];
    __shared__ bool is_last;

    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const uint32_t L = a.L;
    const double cphi = a.cphi, sphi = a.sphi;
    for (int k = threadIdx.x; k <= kTabN; k += blockDim.x) {      // (cos, sin)(h_k - phi), once per CTA and sweep
        const double2 cs = __ldg(a.sincos_tab + k);
        const double cr = __fma_rn(cs.x, cphi, cs.y * sphi), sr = __fma_rn(cs.y, cphi, -(cs.x * sphi));
        if constexpr (kObs) reinterpret_cast<double2 *>(smem_raw)[k] = make_double2(cr, sr);
        else reinterpret_cast<float2 *>(smem_raw)[k] = make_float2(__double2float_rn(cr), __double2float_rn(sr));
    }
    const uint32_t tab_adj = (uint32_t)__cvta_generic_to_shared(smem_raw)
                             - __float_as_uint(kTabMagic) * BondsEntry<kObs>::bytes;
    pdl_wait();              // the rotation above reads only the static table: it ran under the previous kernel's tail
    pdl_launch_next();
    __syncthreads();

    // beta: a kernel argument, or (PCC) the controller's; only its two fp32 derivatives stay in registers
    auto load_beta = [&]() {
        return a.beta_from_ctl ? *reinterpret_cast<const volatile double *>(&a.ctl->beta) : a.beta;
    };
    float m2b, delta;
    {
        const double beta = load_beta();
        m2b = (float)(-2.0 * beta * 1.4426950408889634);
        delta = filter_delta(beta);
    }

    double aMx = 0, aMy = 0, aCx = 0, aSx = 0, aCy = 0, aSy = 0;
    double aF[8] = {0, 0, 0, 0, 0, 0, 0, 0};   // kFourier: Fx[0..3], Fy[0..3]
    uint32_t nbx = 0, nby = 0;

    const uint32_t strips_x = L / TW;
    const uint32_t nstrips = strips_x * ((kSlab ? a.rows : L) / RS);
    // slab: the quad index (Philox counter) is that of the whole lattice; the bond bytes are addressed with it from a
    // base moved back by the slab's first quad
    uint8_t *const bonds_g = kSlab ? a.bonds - (((uint64_t)a.y_off * L) >> 2) : a.bonds;
    for (uint32_t strip = blockIdx.x * NW + warp; strip < nstrips; strip += gridDim.x * NW) {
        const uint32_t sy = strip / strips_x, sx = strip - sy * strips_x;
        const uint32_t y0 = sy * RS;
        const uint32_t xl = sx * TW + lane * VEC;
        // halo column (right neighbour of the strip's last column), one lane per row
        __syncwarp();
        if (lane < RS) {
            uint32_t xh = sx * TW + TW;
            if (xh >= L) xh = 0;
            const float th = __ldg(a.theta + (size_t)(y0 + lane) * L + xh);
            double s = 0, c = 0;
            float g = 0;
            site_eval<kBonds, kObs>(th, tab_adj, g, c, s);
            if constexpr (kObs) { h_c[warp][lane] = c; h_s[warp][lane] = s; }
            if constexpr (kBonds) h_g[warp][lane] = g;
            if constexpr (kFourier) {
                double sk, ck;
                sincospi(2.0 * (double)(y0 + lane) / (double)L, &sk, &ck);
                h_ky[warp][lane] = make_double2(ck, sk);
            }
        }
        __syncwarp();
        double colC[VEC], colS[VEC];             // kFourier: column sums over the strip's rows
#pragma unroll
        for (int v = 0; v < VEC; ++v) { colC[v] = 0.0; colS[v] = 0.0; }

        // two register sets (A, B) alternate as "row being finished" and "row below": no copies.  The raw
        // angles of rows r+1 and r+2 are in flight while row r is evaluated (a set is reloaded as soon as
        // its angles are split)
        float tA[VEC], tB[VEC], gA[VEC], gB[VEC];
        double cA[VEC], sA[VEC], cB[VEC], sB[VEC];
        // running addresses (one 64-bit add per row each): quad index of the lane's first site in the row
        // being finished (Philox counter, bond byte), and the row to load next; only the y-halo row of the
        // lattice's last strip row wraps
        uint64_t quad = ((uint64_t)((kSlab ? a.y_off : 0u) + y0) * L + xl) >> 2;
        const float *nxt = a.theta + (size_t)y0 * L + xl;
        const float *halo_row = a.theta + (!kSlab && y0 + RS == L ? (size_t)0 : (size_t)(y0 + RS) * L) + xl;
        load_vec<VEC, true>(nxt, tA);
        nxt += L;
        load_vec<VEC, true>(RS == 1 ? halo_row : nxt, tB);
        nxt += L;
#pragma unroll
        for (int v = 0; v < VEC; ++v) site_eval<kBonds, kObs>(tA[v], tab_adj, gA[v], cA[v], sA[v]);
        load_vec<VEC, true>(RS == 2 ? halo_row : nxt, tA);
        nxt += L;
        // finishes row r-1 (evaluated, in pc/ps/pg): its x bonds, and its y bonds with row r, whose
        // raw angles are in ct and whose (cos, sin, sigma) land in c/s/g; then ct is reloaded with row r+2
        auto step = [&](int r, const double (&pc)[VEC], const double (&ps)[VEC], const float (&pg)[VEC],
                        float (&ct)[VEC], double (&c)[VEC], double (&s)[VEC], float (&g)[VEC]) {
#pragma unroll
            for (int v = 0; v < VEC; ++v) site_eval<kBonds, kObs>(ct[v], tab_adj, g[v], c[v], s[v]);
            if (r + 2 <= RS) {
                load_vec<VEC, true>(r + 2 == RS ? halo_row : nxt, ct);
                nxt += L;
            }
            const uint32_t gy = y0 + r - 1;                 // global row being finished
            double cn = 0, sn = 0;
            float gn = 0;
            if constexpr (kObs) {
                cn = __shfl_down_sync(0xffffffffu, pc[0], 1);
                sn = __shfl_down_sync(0xffffffffu, ps[0], 1);
                if (lane == 31) { cn = h_c[warp][r - 1]; sn = h_s[warp][r - 1]; }
            }
            if constexpr (kBonds) {
                gn = __shfl_down_sync(0xffffffffu, pg[0], 1);
                if (lane == 31) gn = h_g[warp][r - 1];
            }
            // leading 16 bits of the 2 VEC uniforms: word j of call A of the quad serves site 4q+j
            // (x: low half, y: high half); the trailing bits (call B) are drawn only on a close call
            uint32_t wa[VEC];
            if constexpr (kBonds) {
                const U4 w = philox4x32_10_rk((uint32_t)quad, (uint32_t)(quad >> 32), a.t, TAG_BOND, a.rk);
                if constexpr (VEC == 4) { wa[0] = w.x; wa[1] = w.y; wa[2] = w.z; wa[3] = w.w; }
                else { const bool up = (xl & 2u) != 0; wa[0] = up ? w.z : w.x; wa[1] = up ? w.w : w.y; }
            }
            uint32_t xn = 0, yn = 0;
            float dmin = 3.0e38f;
#pragma unroll
            for (int v = VEC - 1; v >= 0; --v) {
                if constexpr (kObs) {
                    const double c2 = (v + 1 < VEC) ? pc[(v + 1) % VEC] : cn;
                    const double s2 = (v + 1 < VEC) ? ps[(v + 1) % VEC] : sn;
                    if constexpr (kFourier) { colC[v] += pc[v]; colS[v] += ps[v]; }
                    else { aMx += pc[v]; aMy += ps[v]; }
                    aCx = __fma_rn(pc[v], c2, aCx);
                    aCx = __fma_rn(ps[v], s2, aCx);
                    aSx = __fma_rn(ps[v], c2, aSx);
                    aSx = __fma_rn(-pc[v], s2, aSx);
                    aCy = __fma_rn(pc[v], c[v], aCy);
                    aCy = __fma_rn(ps[v], s[v], aCy);
                    aSy = __fma_rn(ps[v], c[v], aSy);
                    aSy = __fma_rn(-pc[v], s[v], aSy);
                }
                if constexpr (kBonds) {
                    const float g2 = (v + 1 < VEC) ? pg[(v + 1) % VEC] : gn;
                    const float gs = pg[v] * m2b;
                    const float dx = bond_filter(gs, g2, wa[v] << 7);
                    const float dy = bond_filter(gs, g[v], wa[v] >> 9);
                    dmin = fminf(dmin, fminf(fabsf(dx), fabsf(dy)));
                    xn = __funnelshift_l(__float_as_uint(dx), xn, 1);         // (xn << 1) | sign(dx): active iff d < 0
                    yn = __funnelshift_l(__float_as_uint(dy), yn, 1);
                }
            }
            if constexpr (kFourier) {
                double rc = pc[0], rs = ps[0];
#pragma unroll
                for (int v = 1; v < VEC; ++v) { rc += pc[v]; rs += ps[v]; }
                const double2 ky = h_ky[warp][r - 1];
                aF[4] = __fma_rn(rc, ky.x, aF[4]); aF[5] = __fma_rn(rc, ky.y, aF[5]);
                aF[6] = __fma_rn(rs, ky.x, aF[6]); aF[7] = __fma_rn(rs, ky.y, aF[7]);
            }
            if constexpr (kBonds) {
                if (!(dmin > delta)) {                   // rare: some decision of this lane is too close to call (or NaN)
                    BondCtx bcx;
                    bcx.phi = a.phi;
                    bcx.beta = load_beta();
                    bcx.m2b = m2b;
                    bcx.delta = delta;
                    bcx.fallback_counter = &a.ctl->fallback_count;
                    RowSigma<VEC> rsg;
#pragma unroll
                    for (int v = 0; v < VEC; ++v) { rsg.pg[v] = pg[v]; rsg.g[v] = g[v]; }
                    rsg.gn = gn;
                    const uint32_t fixed = bonds_fix<VEC>(a.theta, L, kSlab ? 0u : L, a.seed_lo, a.seed_hi, a.t, bcx, quad, gy, xl, rsg, xn | (yn << 8));
                    xn = fixed & 0xffu;
                    yn = fixed >> 8;
                }
                nbx += __popc(xn);
                nby += __popc(yn);
                if constexpr (VEC == 4) {
                    bonds_g[quad] = (uint8_t)(xn | (yn << 4));
                } else {
                    // two lanes share a byte: even lane holds sites 4k,4k+1; odd lane 4k+2,4k+3
                    const uint32_t mine = xn | (yn << 4);
                    const uint32_t other = __shfl_xor_sync(0xffffffffu, mine, 1);
                    if ((lane & 1) == 0) bonds_g[quad] = (uint8_t)(mine | (other << 2));
                }
            }
            quad += L >> 2;
        };
        static_assert(RS % 2 == 0, "the row loop is unrolled by two");
#pragma unroll 1
        for (int r = 1; r <= RS; r += 2) {
            step(r, cA, sA, gA, tB, cB, sB, gB);
            step(r + 1, cB, sB, gB, tA, cA, sA, gA);
        }
        if constexpr (kFourier) {
            double sk, ck;
            sincospi(2.0 * (double)xl / (double)L, &sk, &ck);
#pragma unroll
            for (int v = 0; v < VEC; ++v) {
                aMx += colC[v]; aMy += colS[v];
                aF[0] = __fma_rn(colC[v], ck, aF[0]); aF[1] = __fma_rn(colC[v], sk, aF[1]);
                aF[2] = __fma_rn(colS[v], ck, aF[2]); aF[3] = __fma_rn(colS[v], sk, aF[3]);
                const double cn = __fma_rn(ck, a.ck1, -sk * a.sk1);      // next column: rotate by 2 pi / L
                sk = __fma_rn(sk, a.ck1, ck * a.sk1);
                ck = cn;
            }
        }
    }

    // ---- per-CTA partial sums, fixed tree ----
    double acc[NS];
    acc[0] = aMx; acc[1] = aMy; acc[2] = aCx; acc[3] = aSx; acc[4] = aCy; acc[5] = aSy;
    if constexpr (kFourier) {
#pragma unroll
        for (int k = 0; k < 8; ++k) acc[6 + k] = aF[k];
    }
    if constexpr (kObs) {
#pragma unroll
        for (int k = 0; k < NS; ++k) acc[k] = warp_sum(acc[k]);
    }
    unsigned long long cbx = warp_sum_u64(nbx), cby = warp_sum_u64(nby);
    if (lane == 0) {
        if constexpr (kObs) {
#pragma unroll
            for (int k = 0; k < NS; ++k) red[warp][k] = acc[k];
        }
        redc[warp][0] = cbx; redc[warp][1] = cby;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double tot[NS];
        for (int k = 0; k < NS; ++k) tot[k] = 0.0;
        unsigned long long c0 = 0, c1 = 0;
        for (int w = 0; w < NW; ++w) {
            if constexpr (kObs) for (int k = 0; k < NS; ++k) tot[k] += red[w][k];
            c0 += redc[w][0]; c1 += redc[w][1];
        }
        double *p = a.partials + (size_t)blockIdx.x * kPartialStride;
        if constexpr (kObs) for (int k = 0; k < NS; ++k) p[k] = tot[k];
        p[14] = __longlong_as_double((long long)c0);
        p[15] = __longlong_as_double((long long)c1);
        __threadfence();
        const unsigned int ticket = atomicAdd(&a.ctl->ticket, 1u);
        is_last = (ticket == gridDim.x - 1);
    }
    __syncthreads();
    if (!is_last) return;

    // ---- finalize (S8): the last CTA reduces the partials in a fixed order ----
    __threadfence();
    {
        for (int k = 0; k < NS; ++k) acc[k] = 0.0;
        unsigned long long c0 = 0, c1 = 0;
        for (uint32_t b = threadIdx.x; b < gridDim.x; b += blockDim.x) {
            const double *p = a.partials + (size_t)b * kPartialStride;
            if constexpr (kObs) for (int k = 0; k < NS; ++k) acc[k] += __ldcg(p + k);
            c0 += (unsigned long long)__double_as_longlong(__ldcg(p + 14));
            c1 += (unsigned long long)__double_as_longlong(__ldcg(p + 15));
        }
        if constexpr (kObs) for (int k = 0; k < NS; ++k) acc[k] = warp_sum(acc[k]);
        c0 = warp_sum_u64(c0); c1 = warp_sum_u64(c1);
        __syncthreads();
        if (lane == 0) {
            if constexpr (kObs) for (int k = 0; k < NS; ++k) red[warp][k] = acc[k];
            redc[warp][0] = c0; redc[warp][1] = c1;
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            double tot[NS];
            for (int k = 0; k < NS; ++k) tot[k] = 0.0;
            unsigned long long b0 = 0, b1 = 0;
            for (int w = 0; w < NW; ++w) {
                if constexpr (kObs) for (int k = 0; k < NS; ++k) tot[k] += red[w][k];
                b0 += redc[w][0]; b1 += redc[w][1];
            }
            // sums that are linear in (cos, sin)(theta - phi): back to the lattice frame,
            // cos theta = c cos phi - s sin phi, sin theta = s cos phi + c sin phi
            auto unrotate = [&](double &vc, double &vs) {
                const double rc = __fma_rn(vc, cphi, -(vs * sphi)), rs = __fma_rn(vs, cphi, vc * sphi);
                vc = rc; vs = rs;
            };
            if constexpr (kObs) unrotate(tot[0], tot[1]);
            if constexpr (kFourier) {
                unrotate(tot[6], tot[8]); unrotate(tot[7], tot[9]);       // Fx = (c cos kx, c sin kx, s cos kx, s sin kx)
                unrotate(tot[10], tot[12]); unrotate(tot[11], tot[13]);
                if (a.obs_fill) {
                    xy_fourier *f = a.fring + (a.t % a.ring_cap);   // record of T = t (the incoming state)
                    f->sweep = (uint64_t)a.t;
                    for (int k = 0; k < 4; ++k) { f->Fx[k] = tot[6 + k]; f->Fy[k] = tot[10 + k]; }
                }
            }
            const double N = (double)L * (double)L;
            if constexpr (kObs) {
                if (a.obs_fill) {
                    xy_obs *o = a.ring + (a.t % a.ring_cap);         // record of T = t (the incoming state)
                    o->Mx = tot[0]; o->My = tot[1]; o->Cx = tot[2]; o->Sx = tot[3]; o->Cy = tot[4]; o->Sy = tot[5];
                    o->E = -(tot[2] + tot[4]);
                }
                if (a.feed_pcc) {
                    double chik = 0.0;                                  // (|F_x|^2 + |F_y|^2) / (2 N), Eq. 9 at k = 2 pi / L
                    if constexpr (kFourier) {
                        for (int k = 6; k < 14; ++k) chik = __fma_rn(tot[k], tot[k], chik);
                        chik = __ddiv_rn(chik, __dmul_rn(2.0, N));
                    }
                    pcc_feed(a.ctl, N, tot[2], tot[3], tot[4], tot[5], tot[0], tot[1], chik);
                }
            }
            if constexpr (kBonds) {
                xy_obs *o = a.ring + ((a.t + 1u) % a.ring_cap);  // record of T = t+1, completed later
                o->sweep = (uint64_t)a.t + 1u;
                o->beta = load_beta();
                const double qnan = __longlong_as_double(0x7ff8000000000000LL);
                o->E = qnan; o->Mx = qnan; o->My = qnan; o->Cx = qnan; o->Sx = qnan; o->Cy = qnan; o->Sy = qnan;
                o->n_bonds_x = b0; o->n_bonds_y = b1; o->n_clusters = 0;
                if (a.fring) {                                   // XY_FLAG_FOURIER: the same for the structure-factor record of T = t+1
                    xy_fourier *f = a.fring + ((a.t + 1u) % a.ring_cap);
                    f->sweep = (uint64_t)a.t + 1u;
                    for (int k = 0; k < 4; ++k) { f->Fx[k] = qnan; f->Fy[k] = qnan; }
                }
            }
            a.ctl->ticket = 0;
            __threadfence();
        }
    }
}

// ---------------------------------------------------------------------------------------------
// k_label (S3): tile-local labeling from the packed bond bits; integer only, bit-parallel.
// One CTA per TW x TH tile, TW = 32*WPR; thread (r, w) owns WORD w of row r: 32 sites whose x and
// y bond bits sit in one register each.  The union-find runs over RUNS (maximal chains of x
// bonds inside the tile); a run is named by the tile-local index of its first site.
//   prep    X, Y words from the nibble-packed bytes; S = run-start bits; LL = last run start to
//           the left of the word (runs may span words).
//   union   every y bond that is not redundant (its left neighbour is joined to it in both rows
//           and has its own y bond) unites the runs above and below: lock-free min-link union in
//           shared memory, all rows at once.
//   flatten every run start finds its root and stores it; a bit per site says "tile-local root"
//           (rootmask, read by k_flip).
//   emit    label of a site = global index of the root of its run, 4 sites per thread, coalesced.
// Bonds that leave the tile are left to k_merge.
// ---------------------------------------------------------------------------------------------
template <int WPR, int TH>
constexpr size_t k_label_smem_bytes() { return (size_t)(32 * WPR) * TH * 2 + (size_t)TH * WPR * 12 + (size_t)(32 * WPR) * TH + 32; }

__device__ __forceinline__ uint32_t nib_lo16(uint32_t v)      // low nibbles of 4 bytes -> 16 bits
{
    uint32_t t = v & 0x0F0F0F0Fu;
    t = (t | (t >> 4)) & 0x00FF00FFu;
    return (t | (t >> 8)) & 0xFFFFu;
}

// The tile-local union-find stores parents as 16-bit BYTE offsets into parent[] (index * 2; a tile has
// at most 2^15 sites): a hop is one shared load at [value + base] with no address arithmetic, and the
// array is half the size of 32-bit indices (shared memory bounds the CTAs per SM of k_label).  Order
// and equality are those of the indices.
__device__ __forceinline__ uint32_t pload(const unsigned char *pb, uint32_t off)
{
    return *reinterpret_cast<const volatile uint16_t *>(pb + off);
}

// atomicMin on a 16-bit entry (compare-and-swap on its 32-bit word); returns the old entry
__device__ __forceinline__ uint32_t pmin(unsigned char *pb, uint32_t off, uint32_t val)
{
    uint32_t *word = reinterpret_cast<uint32_t *>(pb + (off & ~3u));
    const uint32_t sh = (off & 2u) * 8u;
    uint32_t old = *reinterpret_cast<volatile uint32_t *>(word);
    for (;;) {
        const uint32_t cur = (old >> sh) & 0xffffu;
        if (cur <= val) return cur;
        const uint32_t prev = atomicCAS(word, old, (old & ~(0xffffu << sh)) | (val << sh));
        if (prev == old) return cur;
        old = prev;
    }
}

// find with path halving: every node on the way is re-pointed to its grandparent.  Racing writers
// only ever replace a parent by an ancestor, so concurrent finds and min-links stay correct.
__device__ __forceinline__ uint32_t sfind_h(unsigned char *pb, uint32_t a)
{
    uint32_t r = pload(pb, a);
    while (r != a) {
        const uint32_t g = pload(pb, r);
        if (g == r) return r;
        *reinterpret_cast<volatile uint16_t *>(pb + a) = (uint16_t)g;
        a = g;
        r = pload(pb, a);
    }
    return a;
}

// min-link union of the components of a and b (any nodes; byte offsets)
__device__ __forceinline__ void sunion_v(unsigned char *pb, uint32_t a, uint32_t b)
{
    for (;;) {
        a = sfind_h(pb, a);
        b = sfind_h(pb, b);
        if (a == b) return;
        const uint32_t hi = a > b ? a : b, lo = a > b ? b : a;
        const uint32_t old = pmin(pb, hi, lo);
        if (old == hi) return;
        a = old;                                   // hi was linked meanwhile: go on from its new parent
        b = lo;
    }
}

template <int WPR, int TH, typename LabelT>
__global__ void __launch_bounds__(WPR * TH, 1536 / (WPR * TH))
k_label(const SweepArgs a)
{
    constexpr int TW = 32 * WPR, NT = WPR * TH;
    constexpr uint32_t LCAP = TW * TH / 2;           // entries of the wave lists: half the worst case (every y bond uniting)
    constexpr uint32_t NONE = 0xffffffffu;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    static_assert(TW * TH <= 32768, "16-bit byte offsets");
    uint16_t *parent = reinterpret_cast<uint16_t *>(smem_raw);                       // [TW*TH]
    uint32_t (*Xs)[WPR] = reinterpret_cast<uint32_t (*)[WPR]>(smem_raw + (size_t)TW * TH * 2);
    uint32_t (*Ss)[WPR] = reinterpret_cast<uint32_t (*)[WPR]>(smem_raw + (size_t)TW * TH * 2 + (size_t)TH * WPR * 4);
    uint32_t (*LLs)[WPR] = reinterpret_cast<uint32_t (*)[WPR]>(smem_raw + (size_t)TW * TH * 2 + (size_t)TH * WPR * 8);
    uint16_t *wlist = reinterpret_cast<uint16_t *>(smem_raw + (size_t)TW * TH * 2 + (size_t)TH * WPR * 12);           // per-wave lists of uniting y bonds (upper site)
    uint32_t *wcnt = reinterpret_cast<uint32_t *>(smem_raw + (size_t)TW * TH * 2 + (size_t)TH * WPR * 12 + (size_t)TW * TH);   // [8] bonds in the list of wave j

    const uint32_t L = a.L;
    LabelT *labels = reinterpret_cast<LabelT *>(a.labels);
    const uint32_t tile = blockIdx.x;
    const uint32_t ty = tile / a.tiles_x, tx = tile - ty * a.tiles_x;
    const uint32_t x0 = tx * TW, y0 = ty * TH;
    const int tid = threadIdx.x;
    const int r = tid / WPR, w = tid % WPR;
    const uint32_t base = r * TW + 32 * w;          // tile-local index of this word's first site

    // ---- prep ----
    pdl_wait();
    pdl_launch_next();
    uint32_t X, Y;
    {
        const size_t i = (size_t)(y0 + r) * L + x0 + 32 * w;
        const uint2 raw = __ldg(reinterpret_cast<const uint2 *>(a.bonds + (i >> 2)));
        X = nib_lo16(raw.x) | (nib_lo16(raw.y) << 16);
        Y = nib_lo16(raw.x >> 4) | (nib_lo16(raw.y >> 4) << 16);
    }
    if (w == WPR - 1) X &= 0x7fffffffu;             // that bond leaves the tile
    if (r == TH - 1) Y = 0u;                        // so do these
    const uint32_t xl = __shfl_up_sync(0xffffffffu, X, 1);
    const uint32_t S = ~((X << 1) | (w > 0 ? xl >> 31 : 0u));
    const uint32_t lastS = S ? base + 31 - __clz(S) : NONE;
    uint32_t LL = NONE;
#pragma unroll
    for (int d = 1; d < WPR; ++d) {
        const uint32_t v = __shfl_up_sync(0xffffffffu, lastS, d);
        if (LL == NONE && d <= w) LL = v;
    }
    Xs[r][w] = X; Ss[r][w] = S; LLs[r][w] = LL;
    if (tid < 8) wcnt[tid] = 0;
    __syncthreads();

    // quad mapping (4 consecutive sites per thread, one row per TW/4 threads): conflict-free 16-byte
    // accesses to parent[] and coalesced label stores
    constexpr int Q = TW / 4, RPP = NT / Q;          // quads per row, rows per pass
    const int q = tid % Q, rq = tid / Q;
    const int wq = q >> 3, o = (q & 7) * 4;

    // ---- parent[site] = first site of its run (a run start points to itself) ----
#pragma unroll 2
    for (int k = 0; k < TH / RPP; ++k) {
        const int row = k * RPP + rq;
        const uint32_t Sq = Ss[row][wq];
        const uint32_t wbase = row * TW + 32 * wq;
        const uint32_t m = Sq & ((2u << o) - 1u);
        uint4 st;
        st.x = (m ? wbase + 31 - __clz(m) : LLs[row][wq]) * 2u;              // byte offsets (see pload)
        st.y = ((Sq >> (o + 1)) & 1u) ? (wbase + o + 1) * 2u : st.x;
        st.z = ((Sq >> (o + 2)) & 1u) ? (wbase + o + 2) * 2u : st.y;
        st.w = ((Sq >> (o + 3)) & 1u) ? (wbase + o + 3) * 2u : st.z;
        *reinterpret_cast<uint2 *>(&parent[wbase + o]) = make_uint2(st.x | (st.y << 16), st.z | (st.w << 16));
    }

    uint32_t need = 0;
    int myj = 0;
    // ---- which y bonds unite two runs: not the redundant ones.  They are sorted into one list per
    //      union wave (below): row r is the upper row of a boundary of wave j = ctz(r + 1) + 1 ----
    {
        const int rb = (r + 1 < TH) ? r + 1 : r;
        const uint32_t J = X & Xs[rb][w] & Y;
        const uint32_t jl = __shfl_up_sync(0xffffffffu, J, 1);
        need = Y & ~((J << 1) | (w > 0 ? jl >> 31 : 0u));
        if (need) {
            myj = __ffs(r + 1);
            const uint32_t cap = LCAP >> myj, off = LCAP - (LCAP >> (myj - 1));
            uint32_t slot = atomicAdd(&wcnt[myj], (uint32_t)__popc(need));
            while (need && slot < cap) {             // what does not fit (lists hold half the worst case) stays with this thread
                const int c = __ffs(need) - 1;
                need &= need - 1;
                wlist[off + slot++] = (uint16_t)(base + c);
            }
        }
    }
    __syncthreads();

    // ---- union, in log2(TH) waves: wave j joins blocks of 2^(j-1) rows pairwise, so every wave
    //      links roots of forests that are already flat and the trees stay shallow.  The bonds of a
    //      wave are dealt out evenly to ALL threads from the wave's list.
    // parent[site] is the site's run start, or (for a run start that was linked already) an ancestor of
    // it: either way a node of the right component to start the finds from
    unsigned char *pb = reinterpret_cast<unsigned char *>(parent);
    auto unite_at = [&](uint32_t site) {
        XY_CHECK(CHK_WLIST, site + TW < (uint32_t)(TW * TH));
        const uint32_t ea = pload(pb, site * 2u), eb = pload(pb, (site + TW) * 2u);
        XY_CHECK(CHK_PARENT, ea < (uint32_t)(TW * TH * 2) && eb < (uint32_t)(TW * TH * 2) && !(ea & 1u) && !(eb & 1u));
        sunion_v(pb, ea, eb);
    };
#pragma unroll 1
    for (int j = 1; (1 << j) <= TH; ++j) {
        const uint32_t n = min(wcnt[j], (uint32_t)(LCAP >> j));
        const uint16_t *lst = wlist + (LCAP - (LCAP >> (j - 1)));
        const uint32_t per = (n + NT - 1) / NT, i1 = min(n, (tid + 1) * per);
        for (uint32_t i = tid * per; i < i1; ++i) unite_at(lst[i]);   // contiguous share: neighbouring bonds mostly join the same runs
        if (myj == j) {
            while (need) {                                            // overflow of the list (dense y bonds): this thread's own
                const int c = __ffs(need) - 1;
                need &= need - 1;
                unite_at(base + c);
            }
        }
        __syncthreads();
    }

    // ---- flatten: ONE pass of parent[i] <- parent[parent[i]] over all entries (fixed cost, no
    //      divergence; the wave order leaves most chains at length <= 2), emit walks what is left.
    //      In place and without a barrier before emit: a racing reader sees an ancestor.
    {
#pragma unroll 2
        for (int k = 0; k < TH / RPP; ++k) {
            const uint32_t i0 = (k * RPP + rq) * TW + 4 * q;
            const uint2 w1 = *reinterpret_cast<const uint2 *>(&parent[i0]);
            uint4 p2;
            p2.x = pload(pb, w1.x & 0xffffu); p2.y = pload(pb, w1.x >> 16);
            p2.z = pload(pb, w1.y & 0xffffu); p2.w = pload(pb, w1.y >> 16);
            *reinterpret_cast<uint2 *>(&parent[i0]) = make_uint2(p2.x | (p2.y << 16), p2.z | (p2.w << 16));
        }
    }

    // ---- emit: label = global index of the root; rootmask bit = "I am the tile-local root" ----
    const LabelT gbase = (LabelT)y0 * L + x0;
#pragma unroll 2
    for (int k = 0; k < TH / RPP; ++k) {
        const int row = k * RPP + rq;
        const uint32_t i0 = row * TW + 4 * q;
        const uint2 rt = *reinterpret_cast<const uint2 *>(&parent[i0]);
        uint32_t root[4] = {rt.x & 0xffffu, rt.x >> 16, rt.y & 0xffffu, rt.y >> 16};
        {
            uint32_t up[4];
#pragma unroll
            for (int v = 0; v < 4; ++v) up[v] = pload(pb, root[v]);
            while (up[0] != root[0] || up[1] != root[1] || up[2] != root[2] || up[3] != root[3]) {   // rare: a longer chain
#pragma unroll
                for (int v = 0; v < 4; ++v) { root[v] = up[v]; up[v] = pload(pb, root[v]); }
            }
        }
        LabelT out[4];
        uint32_t nib = 0;
#pragma unroll
        for (int v = 0; v < 4; ++v) {
            const uint32_t rl = root[v] >> 1;                            // byte offset -> tile-local index
            XY_CHECK(CHK_PARENT, rl <= i0 + v);                         // a root is never after its site
            out[v] = gbase + (LabelT)(rl / TW) * (L - TW) + rl;          // row * L + col with row * TW + col = rl
            nib |= (rl == i0 + v) ? (1u << v) : 0u;
        }
        const size_t gi = (size_t)(y0 + row) * L + x0 + 4 * q;
        LabelT *dst = labels + gi;
        if constexpr (sizeof(LabelT) == 4) {
            *reinterpret_cast<uint4 *>(dst) = make_uint4(out[0], out[1], out[2], out[3]);
        } else {
            *reinterpret_cast<ulonglong2 *>(dst) = make_ulonglong2(out[0], out[1]);
            *reinterpret_cast<ulonglong2 *>(dst + 2) = make_ulonglong2(out[2], out[3]);
        }
        const uint32_t hi = __shfl_down_sync(0xffffffffu, nib, 1);
        if ((q & 1) == 0) reinterpret_cast<uint8_t *>(a.rootmask)[gi >> 3] = (uint8_t)(nib | (hi << 4));
    }
}

// ---------------------------------------------------------------------------------------------
// k_merge: unions across tile edges.  Thread e of tile k: e < TH -> right edge, row e;
// else bottom edge, column e - TH.
// ---------------------------------------------------------------------------------------------
template <int TW, int TH, typename LabelT>
__global__ void __launch_bounds__(256)
k_merge(const SweepArgs a)
{
    pdl_wait();
    pdl_launch_next();
    const uint32_t L = a.L;
    LabelT *labels = reinterpret_cast<LabelT *>(a.labels);
    const uint64_t total = (uint64_t)a.ntiles * (TW + TH);
    const uint64_t total_up = (total + 31u) & ~(uint64_t)31u;                  // whole warps stay in the loop (shuffles)
    for (uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; k < total_up; k += (uint64_t)gridDim.x * blockDim.x) {
        bool active = false;
        LabelT la = 0, lb = 0;
        if (k < total) {
            const uint32_t tile = (uint32_t)(k / (TW + TH));
            const uint32_t e = (uint32_t)(k - (uint64_t)tile * (TW + TH));
            const uint32_t ty = tile / a.tiles_x, tx = tile - ty * a.tiles_x;
            uint32_t x, y, x2, y2, bit;
            if (e < TH) {
                x = tx * TW + TW - 1; y = ty * TH + e;
                x2 = x + 1 == L ? 0 : x + 1; y2 = y;
                bit = 3;                                   // bx of the 4th site of its byte
            } else {
                x = tx * TW + (e - TH); y = ty * TH + TH - 1;
                x2 = x; y2 = y + 1 == a.rows ? 0 : y + 1;
                bit = 4 + (x & 3u);
            }
            const size_t i = (size_t)y * L + x;
            const bool cut = a.open_y && e >= TH && y + 1 == a.rows;      // slab: that bond crosses into the next slab (stitch)
            if (!cut && ((a.bonds[i >> 2] >> bit) & 1u)) {
                active = true;
                la = gload(labels + i);
                lb = gload(labels + (size_t)y2 * L + x2);
            }
        }
        // the edge bonds of a tile mostly join the same few pairs of tile-local components: of all
        // lanes of the warp with the same (la, lb) only the lowest does the union
        const uint32_t act = __ballot_sync(0xffffffffu, active);
        const uint32_t same = __match_any_sync(0xffffffffu, la) & __match_any_sync(0xffffffffu, lb) & act;
        const bool dup = (same & ((1u << (threadIdx.x & 31)) - 1u)) != 0;
        if (active && !dup) gunion<LabelT>(labels, la, lb);
    }
}

// ---------------------------------------------------------------------------------------------
// k_flip (S5 + S6): coin of every site's cluster, reflection, cluster count.  One CTA per
// TW x TH tile (the tiles of k_label), 4 consecutive sites x TH/RPP rows per thread.
//   coins   one Philox call per tile row gives the coins of all 128 labels of that row
//           (coin of label rho = bit rho mod 128 of the call keyed by rho div 128).
//   roots   a tile-local root that still is a global root (label == own index) takes its coin
//           from that table; one that k_merge linked elsewhere is queued, and the queue is
//           worked off densely: chase to the global root (read-only: the forest is final),
//           one Philox call for that root.  Each tile root publishes its coin in shared memory.
//   sites   every other site reads the coin published by its tile root (its label), reflects,
//           and rows in which nothing flipped are not written back.
// ---------------------------------------------------------------------------------------------
template <int WPR, int TH, typename LabelT, bool kSlab = false>
__global__ void __launch_bounds__(WPR * TH, (sizeof(LabelT) == 4 && !kSlab ? 1536 : 1024) / (WPR * TH))
k_flip(const SweepArgs a)
{
    constexpr int TW = 32 * WPR, NT = WPR * TH;
    constexpr int Q = TW / 4, RPP = NT / Q, NP = TH / RPP;
    __shared__ uint32_t cbits[TH * WPR];             // coin of the tile root at tile-local index loc: bit loc
    __shared__ uint16_t queue[2 * (TW + TH)];        // merged tile roots: each owns a component that touches the tile edge, so at most one per edge site
    __shared__ float4 th_s[NP * NT];                 // the tile's angles, staged by cp.async while the label phases run
    __shared__ uint32_t nqueue;
    __shared__ unsigned long long sc[NT / 32];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t L = a.L;
    const LabelT *labels = reinterpret_cast<const LabelT *>(a.labels);
    const uint32_t tile = blockIdx.x;
    const uint32_t ty = tile / a.tiles_x, tx = tile - ty * a.tiles_x;
    const uint32_t x0 = tx * TW, y0 = ty * TH;
    const int q = tid % Q, rq = tid / Q;
    const LabelT gbase = (LabelT)y0 * L + x0;

    // theta of my 4 x NP sites -> shared memory, asynchronously (no registers held): its DRAM latency
    // hides behind the label phases; each thread later reads back exactly what it copied
#pragma unroll
    for (int k = 0; k < NP; ++k) {
        const size_t i = (size_t)(y0 + k * RPP + rq) * L + x0 + 4 * q;
        const uint32_t dst = (uint32_t)__cvta_generic_to_shared(&th_s[k * NT + tid]);
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(a.theta + i) : "memory");
    }
    asm volatile("cp.async.commit_group;" ::: "memory");

    if (tid == 0) nqueue = 0;
    const uint64_t goff = kSlab ? (uint64_t)a.y_off * L : 0;      // slab: coins are keyed by the label in the whole lattice (a multiple of 128)
    if (tid < TH) {
        const uint64_t g = (uint64_t)(y0 + tid) * L + x0 + goff;
        const U4 c = rng(a.seed_lo, a.seed_hi, g >> 7, a.t, TAG_FLIP);
        if constexpr (WPR == 4) {
            *reinterpret_cast<uint4 *>(&cbits[tid * 4]) = make_uint4(c.x, c.y, c.z, c.w);
        } else {
            const bool up = (g & 64u) != 0;
            cbits[tid * 2] = up ? c.z : c.x;
            cbits[tid * 2 + 1] = up ? c.w : c.y;
        }
    }

    // theta (final since the previous sweep's k_flip) and the coin rows needed nothing of k_merge
    pdl_wait();
    pdl_launch_next();
    // labels are read twice (here and in the last phase; the second read hits L1/L2) rather than
    // held in registers: few registers, so many CTAs per SM hide the latency of the phases
    auto load_labels = [&](size_t i, LabelT (&lab)[4]) {
        if constexpr (sizeof(LabelT) == 4) {
            const uint4 v = __ldg(reinterpret_cast<const uint4 *>(labels + i));
            lab[0] = v.x; lab[1] = v.y; lab[2] = v.z; lab[3] = v.w;
        } else {
            const ulonglong2 u = __ldg(reinterpret_cast<const ulonglong2 *>(labels + i));
            const ulonglong2 v = __ldg(reinterpret_cast<const ulonglong2 *>(labels + i + 2));
            lab[0] = u.x; lab[1] = u.y; lab[2] = v.x; lab[3] = v.y;
        }
    };
    uint32_t rb = 0;                                 // root bits of my 4 sites in pass k: nibble k
    // ---- tile roots that k_merge linked elsewhere are queued; the others are the clusters ----
    uint32_t merged = 0;
#pragma unroll
    for (int k = 0; k < NP; ++k) {
        const int row = k * RPP + rq;
        const size_t i = (size_t)(y0 + row) * L + x0 + 4 * q;
        LabelT lab[4];
        load_labels(i, lab);
        const uint32_t nib = (__ldg(reinterpret_cast<const uint8_t *>(a.rootmask) + (i >> 3)) >> (i & 4u)) & 15u;
        rb |= nib << (4 * k);
#pragma unroll
        for (int v = 0; v < 4; ++v)
            if (lab[v] != (LabelT)(i + v)) merged |= 1u << (4 * k + v);
    }
    merged &= rb;
    uint32_t ncl = __popc(rb & ~merged);
    __syncthreads();                                 // nqueue = 0 and cbits visible
    while (merged) {
        const int b = __ffs(merged) - 1;
        merged &= merged - 1;
        const uint32_t slot = atomicAdd(&nqueue, 1u);
        XY_CHECK(CHK_QUEUE, slot < (uint32_t)(2 * (TW + TH)));
        queue[slot] = (uint16_t)(((b >> 2) * RPP + rq) * TW + 4 * q + (b & 3));
    }
    __syncthreads();
    {
        const uint32_t nq = nqueue;
        for (uint32_t j = tid; j < nq; j += NT) {
            const uint32_t loc = queue[j];
            const LabelT self = gbase + (LabelT)(loc / TW) * L + (loc % TW);
            LabelT root = __ldg(labels + self);
            uint64_t groot;                                  // canonical label in the whole lattice
            if constexpr (kSlab) {
                // slab: a chain may end in an entry the stitch overrode (kSlabSpecial | k): the root is xroot[k]
                while (!((uint32_t)root & kSlabSpecial)) {
                    const LabelT p = __ldg(labels + root);
                    if (p == root) break;
                    XY_CHECK(CHK_GLABEL, ((uint32_t)p & kSlabSpecial) || p < root);
                    root = p;
                }
                if ((uint32_t)root & kSlabSpecial) {
                    XY_CHECK(CHK_GLABEL, ((uint32_t)root & ~kSlabSpecial) < 2u * L);
                    groot = a.xroot[(uint32_t)root & ~kSlabSpecial];
                    if (groot == (uint64_t)self + goff) ++ncl;   // the cluster's canonical root is this very site
                } else {
                    groot = (uint64_t)root + goff;
                }
            } else {
                LabelT p = __ldg(labels + root);
                while (p != root) { XY_CHECK(CHK_GLABEL, p < root); root = p; p = __ldg(labels + root); }
                groot = (uint64_t)root;
            }
            const U4 c = rng(a.seed_lo, a.seed_hi, groot >> 7, a.t, TAG_FLIP);
            const uint32_t sel = ((uint32_t)groot >> 5) & 3u;
            const uint32_t word = sel == 0 ? c.x : sel == 1 ? c.y : sel == 2 ? c.z : c.w;
            const uint32_t coin = (word >> ((uint32_t)groot & 31u)) & 1u;
            if (coin) atomicOr(&cbits[loc >> 5], 1u << (loc & 31u));
            else atomicAnd(&cbits[loc >> 5], ~(1u << (loc & 31u)));
        }
    }
    __syncthreads();

    // ---- every site takes the coin of its tile root; reflect ----
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    const uint32_t Lm = L - TW;
#pragma unroll
    for (int k = 0; k < NP; ++k) {
        const int row = k * RPP + rq;
        const uint32_t loc0 = row * TW + 4 * q;
        const size_t i = (size_t)(y0 + row) * L + x0 + 4 * q;
        const float4 t4 = th_s[k * NT + tid];
        const float th[4] = {t4.x, t4.y, t4.z, t4.w};
        LabelT lab[4];
        load_labels(i, lab);
        uint32_t coins = 0;
#pragma unroll
        for (int v = 0; v < 4; ++v) {
            const uint32_t d = (uint32_t)(lab[v] - gbase);              // r*L + c, < TH*L <= 2^22
            const uint32_t rr = __umulhi(d, a.Ldiv_mul) >> a.Ldiv_shift;
            const uint32_t loc = ((rb >> (4 * k + v)) & 1u) ? loc0 + v : d - rr * Lm;
            XY_CHECK(CHK_LOC, loc < (uint32_t)(TW * TH));
            coins |= ((cbits[loc >> 5] >> (loc & 31u)) & 1u) << v;
        }
        if (coins) {                                                    // one branch per 4 sites; straight-line inside
            float out[4];
#pragma unroll
            for (int v = 0; v < 4; ++v) {
                const float rf = reflect(th[v], a.A);
                out[v] = ((coins >> v) & 1u) ? rf : th[v];
            }
            *reinterpret_cast<float4 *>(a.theta + i) = make_float4(out[0], out[1], out[2], out[3]);
        }
    }

    unsigned long long c = warp_sum_u64(ncl);
    if (lane == 0) sc[warp] = c;
    __syncthreads();
    if (tid == 0) {
        unsigned long long tot = 0;
        for (int w = 0; w < NT / 32; ++w) tot += sc[w];
        xy_obs *o = a.ring + ((a.t + 1u) % a.ring_cap);
        atomicAdd(reinterpret_cast<unsigned long long *>(&o->n_clusters), tot);
    }
}

// ---------------------------------------------------------------------------------------------
// Small utility kernels (init, export, debug).
// ---------------------------------------------------------------------------------------------
// first: index in the whole lattice of the state's first site (a slab starts at row y_off)
__global__ void k_init_hot(float *theta, uint64_t N, uint64_t first, uint32_t seed_lo, uint32_t seed_hi)
{
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (uint64_t)gridDim.x * blockDim.x) {
        const U4 w = rng(seed_lo, seed_hi, first + i, 0u, TAG_INIT);
        const double frac = (double)(w.x >> 8) * (1.0 / 16777216.0);
        theta[i] = __double2float_rn(__dmul_rn(kTwoPi, frac));
    }
}

// in-place flatten for xy_get_labels: label[i] <- root(i).  Concurrent writes only ever replace
// a parent by an ancestor, so readers still reach the same root.
template <typename LabelT>
__global__ void k_flatten(LabelT *labels, uint64_t N)
{
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (uint64_t)gridDim.x * blockDim.x) {
        const LabelT r = gfind<LabelT>(labels, (LabelT)i);
        labels[i] = r;
    }
}

// Whole-lattice invariants of a flattened labeling (xy_debug_check_labels).  out[0]: label[i] > i;
// out[1]: label[label[i]] != label[i]; out[2] / out[3]: an active x / y bond joins unequal labels
// (periodic wrap included); out[4]: number of roots (label[i] == i).  A labeling with all four
// violation counts zero names every cluster by one of its sites, is constant on clusters, and no
// label is above its site's index.
template <typename LabelT>
__global__ void k_check_labels(const LabelT *labels, const uint8_t *bonds, uint32_t L, unsigned long long *out)
{
    const uint64_t N = (uint64_t)L * L;
    unsigned long long v0 = 0, v1 = 0, v2 = 0, v3 = 0, v4 = 0;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (uint64_t)gridDim.x * blockDim.x) {
        const LabelT l = labels[i];
        if ((uint64_t)l > i) { ++v0; continue; }
        if (labels[l] != l) ++v1;
        if ((uint64_t)l == i) ++v4;
        const uint32_t b = bonds[i >> 2];
        const uint32_t j = (uint32_t)(i & 3u);
        const uint32_t x = (uint32_t)(i % L);
        if ((b >> j) & 1u) {
            const uint64_t r = (x + 1 == L) ? i + 1 - L : i + 1;
            if (labels[r] != l) ++v2;
        }
        if ((b >> (4 + j)) & 1u) {
            const uint64_t d = (i + L >= N) ? i + L - N : i + L;
            if (labels[d] != l) ++v3;
        }
    }
    v0 = warp_sum_u64(v0); v1 = warp_sum_u64(v1); v2 = warp_sum_u64(v2); v3 = warp_sum_u64(v3); v4 = warp_sum_u64(v4);
    if ((threadIdx.x & 31) == 0) {
        if (v0) atomicAdd(out + 0, v0);
        if (v1) atomicAdd(out + 1, v1);
        if (v2) atomicAdd(out + 2, v2);
        if (v3) atomicAdd(out + 3, v3);
        if (v4) atomicAdd(out + 4, v4);
    }
}

template <typename LabelT>
__global__ void k_labels_to_i64(const LabelT *labels, int64_t *out, uint64_t first, uint64_t n)
{
    for (uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (uint64_t)gridDim.x * blockDim.x)
        out[k] = (int64_t)labels[first + k];
}

// packed (nibble) layout -> canonical byte per site: bit0 = bx, bit1 = by
__global__ void k_bonds_unpack(const uint8_t *packed, uint8_t *out, uint64_t first, uint64_t n)
{
    for (uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (uint64_t)gridDim.x * blockDim.x) {
        const uint64_t i = first + k;
        const uint32_t b = packed[i >> 2];
        const uint32_t j = (uint32_t)(i & 3u);
        out[k] = (uint8_t)(((b >> j) & 1u) | (((b >> (4 + j)) & 1u) << 1));
    }
}

__global__ void k_bonds_pack(const uint8_t *canon, uint8_t *packed, uint64_t first_group, uint64_t ngroups)
{
    for (uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; k < ngroups; k += (uint64_t)gridDim.x * blockDim.x) {
        uint32_t b = 0;
        for (int j = 0; j < 4; ++j) {
            const uint32_t c = canon[4 * k + j];
            b |= (c & 1u) << j;
            b |= ((c >> 1) & 1u) << (4 + j);
        }
        packed[first_group + k] = (uint8_t)b;
    }
}

__global__ void k_debug_philox(const uint32_t *ctr, const uint32_t *key, uint32_t *out, size_t n)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const U4 w = philox4x32_10(ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3], key[2 * i], key[2 * i + 1]);
    out[4 * i] = w.x; out[4 * i + 1] = w.y; out[4 * i + 2] = w.z; out[4 * i + 3] = w.w;
}

}  // namespace xy
