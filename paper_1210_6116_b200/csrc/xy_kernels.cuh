// xy_kernels.cuh -- the kernels of one Swendsen-Wang sweep of the 2D XY model on sm_100a.
//
//   k_bonds   (S2, and S7 of the incoming configuration): warps stream strips of the lattice row
//             by row: theta -> fp64 (cos, sin, sigma) per site in registers (table + short Taylor
//             rotation) -> observables, Philox bond draws, filtered bond decisions -> packed bond
//             bits (0.25 B/site).  theta is read once (+ halo); no block barrier in the loop.
//   k_label   (S3): one CTA per TW x TH tile, integer only: run starts by ballot/clz over the
//             x-bond bits, union-find over the runs in shared memory -> provisional label (global
//             index of the tile-local root), written once.
//   k_merge        (S4): one thread per tile-edge bond; atomicMin union-find on the label array.
//   k_flip         (S5+S6): chase each site's label to the cluster's root (minimum site index),
//                  draw the root's coin with Philox, reflect, write theta back.
//   finalize       (S8): the last CTA of k_bonds reduces the per-CTA partial sums in a fixed
//                  order, writes the per-sweep record and advances the PCC controller.
//
// Layouts: theta fp32 row-major i = y*L + x.  labels LabelT (u32 or u64) same indexing.
// bonds packed 2 bits/site: byte (i>>2) holds bx(4k+j) in bit j and by(4k+j) in bit 4+j.
#pragma once
#include "xy_device.cuh"
#include "../../include/xy.h"

namespace xy {

constexpr int kPartialStride = 8;          // doubles per CTA partial record

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
    // misc
    unsigned long long fallback_count;
    unsigned int ticket;          // last-block-done counter of k_bonds
    unsigned int pad;
};

struct SweepArgs {
    float       *theta;
    void        *labels;
    uint8_t     *bonds;
    double      *partials;        // [grid][kPartialStride]
    DevCtl      *ctl;
    xy_obs      *ring;
    uint32_t     ring_cap;
    uint32_t     L;
    uint32_t     tiles_x, ntiles;
    uint32_t     seed_lo, seed_hi;
    uint32_t     t;               // sweep counter of THIS sweep (state before it has T = t sweeps done)
    int          beta_from_ctl;   // 1: read beta from ctl->beta (PCC), 0: use beta
    int          feed_pcc;        // 1: finalize feeds the observables of the incoming state to the controller
    int          obs_fill;        // 1: finalize writes the observables of the incoming state into ring[T]
    double       beta;
    double       phi, cphi, sphi, A;
    const double2 *sincos_tab;    // [257] (cos, sin)(2 pi k / 256), host-computed
};


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
__device__ inline void pcc_feed(DevCtl *c, double N, double Cx, double Sx, double Cy, double Sy)
{
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
        if (c->trace_beta && c->n_dec < c->trace_cap) {
            c->trace_beta[c->n_dec] = c->beta;
            c->trace_bY[c->n_dec] = bY;
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
// ---------------------------------------------------------------------------------------------
constexpr int kTabN = 256;                 // sincos table: entries k = 0..256 at angle 2 pi k / 256

// sin, cos of an fp32 angle in [0, 2pi(1+1e-7)]: table lookup + degree-5/4 Taylor rotation in
// fp64, |error| < 1e-15 (|x| <= pi/256: x^7/5040 = 8e-18, x^6/720 = 5e-15).
__device__ __forceinline__ void sincos_tab(float theta, const double2 *tab, double &s, double &c)
{
    const double t = (double)theta;
    const double kd = __fma_rn(t, 40.743665431525208, 6755399441055744.0);      // 256/(2 pi), round to integer
    const int k = __double2loint(kd);
    const double kf = kd - 6755399441055744.0;
    double x = __fma_rn(-kf, 0.02454369260617026, t);                          // fl64(2 pi)/256, exact scaling
    x = __fma_rn(-kf, 9.5675529620887e-19, x);                                  // (2 pi - fl64(2 pi))/256
    const double2 cs = tab[k];
    const double x2 = x * x;
    const double sx = __fma_rn(x * x2, __fma_rn(x2, 8.3333333333333333e-3, -1.6666666666666667e-1), x);
    const double dc = x2 * __fma_rn(x2, 4.1666666666666667e-2, -0.5);           // cos x - 1
    c = __fma_rn(-cs.y, sx, __fma_rn(cs.x, dc, cs.x));
    s = __fma_rn(cs.x, sx, __fma_rn(cs.y, dc, cs.y));
}

template <int VEC, int RS, bool kBonds>
__global__ void __launch_bounds__(128, 4)
k_bonds(const SweepArgs a)
{
    constexpr int NW = 4;
    constexpr int TW = 32 * VEC;
    static_assert(RS <= 32, "halo column is computed by one lane per row");

    __shared__ double2 tab[kTabN + 1];
    __shared__ double h_c[NW][RS], h_s[NW][RS], h_g[NW][RS];
    __shared__ float h_t[NW][RS];
    __shared__ double red[NW][6];
    __shared__ unsigned long long redc[NW][2];
    __shared__ bool is_last;

    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const uint32_t L = a.L;
    for (int k = threadIdx.x; k <= kTabN; k += blockDim.x) tab[k] = a.sincos_tab[k];
    __syncthreads();

    double beta = a.beta;
    if (a.beta_from_ctl) beta = *reinterpret_cast<const volatile double *>(&a.ctl->beta);
    BondCtx bcx;
    bcx.phi = a.phi;
    bcx.beta = beta;
    bcx.m2b = (float)(-2.0 * beta * 1.4426950408889634);
    bcx.fallback_counter = &a.ctl->fallback_count;
    const double cphi = a.cphi, sphi = a.sphi;

    double aMx = 0, aMy = 0, aCx = 0, aSx = 0, aCy = 0, aSy = 0;
    uint32_t nbx = 0, nby = 0;

    const uint32_t strips_x = L / TW;
    const uint32_t nstrips = strips_x * (L / RS);
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
            double s, c;
            sincos_tab(th, tab, s, c);
            h_t[warp][lane] = th;
            h_c[warp][lane] = c;
            h_s[warp][lane] = s;
            h_g[warp][lane] = __fma_rn(c, cphi, s * sphi);
        }
        __syncwarp();

        float pt[VEC], nt[VEC];
        double pc[VEC], ps[VEC], pg[VEC];
        load_vec<VEC, true>(a.theta + (size_t)y0 * L + xl, pt);
        {
            uint32_t y1 = y0 + 1;
            if (y1 >= L) y1 -= L;
            load_vec<VEC, true>(a.theta + (size_t)y1 * L + xl, nt);
        }
#pragma unroll
        for (int v = 0; v < VEC; ++v) {
            sincos_tab(pt[v], tab, ps[v], pc[v]);
            pg[v] = __fma_rn(pc[v], cphi, ps[v] * sphi);
        }
#pragma unroll 1
        for (int r = 1; r <= RS; ++r) {
            // this iteration finishes row r-1 (held in p*): its x bonds, and its y bonds with row r
            float ct[VEC];
#pragma unroll
            for (int v = 0; v < VEC; ++v) ct[v] = nt[v];
            if (r < RS) {                                   // prefetch row r+1
                uint32_t y2 = y0 + r + 1;
                if (y2 >= L) y2 -= L;
                load_vec<VEC, true>(a.theta + (size_t)y2 * L + xl, nt);
            }
            double c[VEC], s[VEC], g[VEC];
#pragma unroll
            for (int v = 0; v < VEC; ++v) {
                sincos_tab(ct[v], tab, s[v], c[v]);
                g[v] = __fma_rn(c[v], cphi, s[v] * sphi);
            }
            const uint32_t gy = y0 + r - 1;                 // global row being finished
            double cn = __shfl_down_sync(0xffffffffu, pc[0], 1);
            double sn = __shfl_down_sync(0xffffffffu, ps[0], 1);
            double gn = __shfl_down_sync(0xffffffffu, pg[0], 1);
            float tn = __shfl_down_sync(0xffffffffu, pt[0], 1);
            if (lane == 31) { cn = h_c[warp][r - 1]; sn = h_s[warp][r - 1]; gn = h_g[warp][r - 1]; tn = h_t[warp][r - 1]; }
            uint32_t wx[VEC], wy[VEC];
            if constexpr (kBonds) {
#pragma unroll
                for (int v = 0; v < VEC; v += 2) {
                    const uint64_t site = (uint64_t)gy * L + xl + v;
                    const U4 w = rng(a.seed_lo, a.seed_hi, site >> 1, a.t, TAG_BOND);
                    wx[v] = w.x; wy[v] = w.y; wx[v + 1] = w.z; wy[v + 1] = w.w;
                }
            }
            uint32_t xn = 0, yn = 0;
#pragma unroll
            for (int v = 0; v < VEC; ++v) {
                const double c2 = (v + 1 < VEC) ? pc[(v + 1) % VEC] : cn;
                const double s2 = (v + 1 < VEC) ? ps[(v + 1) % VEC] : sn;
                const double g2 = (v + 1 < VEC) ? pg[(v + 1) % VEC] : gn;
                const float t2 = (v + 1 < VEC) ? pt[(v + 1) % VEC] : tn;
                aMx += pc[v];
                aMy += ps[v];
                aCx = __fma_rn(pc[v], c2, aCx);
                aCx = __fma_rn(ps[v], s2, aCx);
                aSx = __fma_rn(ps[v], c2, aSx);
                aSx = __fma_rn(-pc[v], s2, aSx);
                aCy = __fma_rn(pc[v], c[v], aCy);
                aCy = __fma_rn(ps[v], s[v], aCy);
                aSy = __fma_rn(ps[v], c[v], aSy);
                aSy = __fma_rn(-pc[v], s[v], aSy);
                if constexpr (kBonds) {
                    if (bond_decide(pg[v] * g2, wx[v], pt[v], t2, bcx)) xn |= 1u << v;
                    if (bond_decide(pg[v] * g[v], wy[v], pt[v], ct[v], bcx)) yn |= 1u << v;
                }
            }
            if constexpr (kBonds) {
                nbx += __popc(xn);
                nby += __popc(yn);
                if constexpr (VEC == 4) {
                    a.bonds[((size_t)gy * L + xl) >> 2] = (uint8_t)(xn | (yn << 4));
                } else {
                    // two lanes share a byte: even lane holds sites 4k,4k+1; odd lane 4k+2,4k+3
                    const uint32_t mine = xn | (yn << 4);
                    const uint32_t other = __shfl_xor_sync(0xffffffffu, mine, 1);
                    if ((lane & 1) == 0) a.bonds[((size_t)gy * L + xl) >> 2] = (uint8_t)(mine | (other << 2));
                }
            }
#pragma unroll
            for (int v = 0; v < VEC; ++v) { pc[v] = c[v]; ps[v] = s[v]; pg[v] = g[v]; pt[v] = ct[v]; }
        }
    }

    // ---- per-CTA partial sums, fixed tree ----
    aMx = warp_sum(aMx); aMy = warp_sum(aMy); aCx = warp_sum(aCx);
    aSx = warp_sum(aSx); aCy = warp_sum(aCy); aSy = warp_sum(aSy);
    unsigned long long cbx = warp_sum_u64(nbx), cby = warp_sum_u64(nby);
    if (lane == 0) {
        red[warp][0] = aMx; red[warp][1] = aMy; red[warp][2] = aCx;
        red[warp][3] = aSx; red[warp][4] = aCy; red[warp][5] = aSy;
        redc[warp][0] = cbx; redc[warp][1] = cby;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double acc[6] = {0, 0, 0, 0, 0, 0};
        unsigned long long c0 = 0, c1 = 0;
        for (int w = 0; w < NW; ++w) {
            for (int k = 0; k < 6; ++k) acc[k] += red[w][k];
            c0 += redc[w][0]; c1 += redc[w][1];
        }
        double *p = a.partials + (size_t)blockIdx.x * kPartialStride;
        for (int k = 0; k < 6; ++k) p[k] = acc[k];
        p[6] = __longlong_as_double((long long)c0);
        p[7] = __longlong_as_double((long long)c1);
        __threadfence();
        const unsigned int ticket = atomicAdd(&a.ctl->ticket, 1u);
        is_last = (ticket == gridDim.x - 1);
    }
    __syncthreads();
    if (!is_last) return;

    // ---- finalize (S8): the last CTA reduces the partials in a fixed order ----
    __threadfence();
    {
        double acc[6] = {0, 0, 0, 0, 0, 0};
        unsigned long long c0 = 0, c1 = 0;
        for (uint32_t b = threadIdx.x; b < gridDim.x; b += blockDim.x) {
            const double *p = a.partials + (size_t)b * kPartialStride;
            for (int k = 0; k < 6; ++k) acc[k] += __ldcg(p + k);
            c0 += (unsigned long long)__double_as_longlong(__ldcg(p + 6));
            c1 += (unsigned long long)__double_as_longlong(__ldcg(p + 7));
        }
        for (int k = 0; k < 6; ++k) acc[k] = warp_sum(acc[k]);
        c0 = warp_sum_u64(c0); c1 = warp_sum_u64(c1);
        __syncthreads();
        if (lane == 0) {
            for (int k = 0; k < 6; ++k) red[warp][k] = acc[k];
            redc[warp][0] = c0; redc[warp][1] = c1;
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            double tot[6] = {0, 0, 0, 0, 0, 0};
            unsigned long long b0 = 0, b1 = 0;
            for (int w = 0; w < NW; ++w) {
                for (int k = 0; k < 6; ++k) tot[k] += red[w][k];
                b0 += redc[w][0]; b1 += redc[w][1];
            }
            const double N = (double)L * (double)L;
            if (a.obs_fill) {
                xy_obs *o = a.ring + (a.t % a.ring_cap);         // record of T = t (the incoming state)
                o->Mx = tot[0]; o->My = tot[1]; o->Cx = tot[2]; o->Sx = tot[3]; o->Cy = tot[4]; o->Sy = tot[5];
                o->E = -(tot[2] + tot[4]);
            }
            if (a.feed_pcc) pcc_feed(a.ctl, N, tot[2], tot[3], tot[4], tot[5]);
            if constexpr (kBonds) {
                xy_obs *o = a.ring + ((a.t + 1u) % a.ring_cap);  // record of T = t+1, completed later
                o->sweep = (uint64_t)a.t + 1u;
                o->beta = beta;
                const double qnan = __longlong_as_double(0x7ff8000000000000LL);
                o->E = qnan; o->Mx = qnan; o->My = qnan; o->Cx = qnan; o->Sx = qnan; o->Cy = qnan; o->Sy = qnan;
                o->n_bonds_x = b0; o->n_bonds_y = b1; o->n_clusters = 0;
            }
            a.ctl->ticket = 0;
            __threadfence();
        }
    }
}

// ---------------------------------------------------------------------------------------------
// k_label (S3): tile-local labeling from the packed bond bits; integer only.  One CTA per
// TW x TH tile (TW = 32*VEC, TH = R*NW); warp w owns the strip of rows [w*R, (w+1)*R).
//   scan   each warp walks its strip top to bottom, all lanes on the same row: run starts of the
//          row by ballot/clz over the x bits -> parent[]; then every y bond that is not redundant
//          ATTACHES the lower run's fresh root to the upper site's root, which the lane carries
//          in registers: one atomicMin, no find.  Only when the run was already attached
//          elsewhere (two upper components meet) a real union runs.  Row order keeps trees flat.
//   stitch unions across the NW-1 strip boundaries (generic lock-step union).
//   emit   provisional label = global index of the tile-local root (min index in the tile-local
//          component).  Bonds that leave the tile are left to k_merge.
// ---------------------------------------------------------------------------------------------
template <int VEC, int R, int NW>
constexpr size_t k_label_smem_bytes() { return (size_t)(32 * VEC) * (R * NW) * 4 + (size_t)NW * 64; }

template <int VEC, int R, int NW, typename LabelT>
__global__ void __launch_bounds__(NW * 32)
k_label(const SweepArgs a)
{
    constexpr int TW = 32 * VEC, TH = R * NW;
    constexpr uint32_t VMASK = (1u << VEC) - 1u;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    uint32_t *parent = reinterpret_cast<uint32_t *>(smem_raw);                     // [TW*TH]
    uint8_t (*xfirst)[32] = reinterpret_cast<uint8_t (*)[32]>(smem_raw + TW * TH * 4);          // x bits of each strip's first row
    uint8_t (*xlast)[32] = reinterpret_cast<uint8_t (*)[32]>(smem_raw + TW * TH * 4 + NW * 32); // x | y << 4 bits of its last row

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t L = a.L;
    LabelT *labels = reinterpret_cast<LabelT *>(a.labels);
    const uint32_t tile = blockIdx.x;
    const uint32_t ty = tile / a.tiles_x, tx = tile - ty * a.tiles_x;
    const uint32_t x0 = tx * TW, y0 = ty * TH;
    const uint32_t xl = x0 + lane * VEC;

    uint32_t bytes[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        uint32_t b = a.bonds[((size_t)(y0 + warp * R + r) * L + xl) >> 2];
        if constexpr (VEC == 2) b = (b >> ((lane & 1) * 2)) & 0x33u;
        bytes[r] = b;
    }

    // ---- scan ----
    uint32_t rootU[VEC];            // root (as of the previous row) of the VEC sites above
    uint32_t xprev = 0, yprev = 0;  // tile-local x bits and y bits of the previous row
#pragma unroll
    for (int v = 0; v < VEC; ++v) rootU[v] = 0;
#pragma unroll 1
    for (int r = 0; r < R; ++r) {
        const int ly = warp * R + r;
        uint32_t xloc = bytes[0] & VMASK;
        const uint32_t yn = (bytes[0] >> 4) & VMASK;
#pragma unroll
        for (int k = 0; k + 1 < R; ++k) bytes[k] = bytes[k + 1];                 // rotate (keeps indices static)
        if (lane == 31) xloc &= ~(1u << (VEC - 1));                              // that bond leaves the tile
        if (r == 0) xfirst[warp][lane] = (uint8_t)xloc;
        // run starts of this row
        const uint32_t through = __ballot_sync(0xffffffffu, xloc == VMASK);
        const uint32_t stop = ~through & ((1u << lane) - 1u);                    // lanes below me that break the run
        const int lp = stop ? 31 - __clz(stop) : 0;
        const uint32_t nib = __shfl_sync(0xffffffffu, xloc, lp);
        uint32_t s0 = 0;
        if (stop) s0 = lp * VEC + (31 - __clz(~nib & VMASK)) + 1;
        uint32_t start[VEC];
        start[0] = ly * TW + s0;
#pragma unroll
        for (int v = 1; v < VEC; ++v)
            start[v] = ((xloc >> (v - 1)) & 1u) ? start[v - 1] : (uint32_t)(ly * TW + lane * VEC + v);
        if constexpr (VEC == 4)
            *reinterpret_cast<uint4 *>(&parent[ly * TW + lane * 4]) = make_uint4(start[0], start[1], start[2], start[3]);
        else
            *reinterpret_cast<uint2 *>(&parent[ly * TW + lane * 2]) = make_uint2(start[0], start[1]);
        __syncwarp();
        if (r > 0) {
            // a y bond is redundant if the left neighbour is joined to me in both rows and has its own y bond
            uint32_t dup = (xprev & xloc & yprev) << 1;
            const uint32_t packed = xprev & xloc & yprev;
            const uint32_t left = __shfl_up_sync(0xffffffffu, packed, 1);
            if (lane > 0) dup |= (left >> (VEC - 1)) & 1u;
            const uint32_t need = yprev & ~dup & VMASK;
            // attach: the lower run's root takes the upper root unless it already has a smaller one
            uint32_t fail = 0, other[VEC];
#pragma unroll
            for (int v = 0; v < VEC; ++v) {
                other[v] = 0;
                if ((need >> v) & 1u) {
                    const uint32_t old = atomicMin(&parent[start[v]], rootU[v]);
                    if (old != start[v] && old != rootU[v]) { fail |= 1u << v; other[v] = old; }
                }
            }
            // two upper components met in one lower run: real union (rare)
            if (__any_sync(0xffffffffu, fail != 0)) {
#pragma unroll
                for (int v = 0; v < VEC; ++v)
                    if ((fail >> v) & 1u) sunion(parent, other[v], rootU[v]);
            }
            __syncwarp();
        }
        // roots of this row's sites for the next row (one extra hop against staleness)
#pragma unroll
        for (int v = 0; v < VEC; ++v) {
            const uint32_t p1 = (v > 0 && start[v] == start[v - 1]) ? rootU[v - 1] : parent[parent[start[v]]];
            rootU[v] = p1;
        }
        xprev = xloc;
        yprev = yn;
    }

    // ---- stitch: strip boundaries IN ORDER, by one warp.  When boundary w is processed the strips
    //      0..w are already one forest whose roots are final for those strips, so every root of
    //      strip w+1 links straight to a final root: chains stay site -> run start -> strip root -> root.
    xlast[warp][lane] = (uint8_t)(xprev | (yprev << 4));
    __syncthreads();
    if (warp == 0) {
#pragma unroll 1
        for (int w = 0; w + 1 < NW; ++w) {
            const uint32_t bu = xlast[w][lane], xu = bu & VMASK, yu = bu >> 4;
            const uint32_t xd = xfirst[w + 1][lane];
            const uint32_t packed = xu & xd & yu;
            uint32_t dup = packed << 1;
            const uint32_t left = __shfl_up_sync(0xffffffffu, packed, 1);
            if (lane > 0) dup |= (left >> (VEC - 1)) & 1u;
            const uint32_t need = yu & ~dup & VMASK;
            const uint32_t above = (w * R + R - 1) * TW + lane * VEC;
#pragma unroll
            for (int v = 0; v < VEC; ++v)
                if ((need >> v) & 1u) sunion(parent, parent[above + v], parent[above + TW + v]);
            __syncwarp();
        }
    }
    __syncthreads();

    // ---- emit: provisional labels (three hops unrolled for all VEC sites, then the rare rest) ----
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int ly = warp * R + r;
        uint32_t p0[VEC], p1[VEC];
        if constexpr (VEC == 4) {
            const uint4 q = *reinterpret_cast<const uint4 *>(&parent[ly * TW + lane * 4]);
            p0[0] = q.x; p0[1] = q.y; p0[2] = q.z; p0[3] = q.w;
        } else {
            const uint2 q = *reinterpret_cast<const uint2 *>(&parent[ly * TW + lane * 2]);
            p0[0] = q.x; p0[1] = q.y;
        }
#pragma unroll
        for (int v = 0; v < VEC; ++v) p1[v] = parent[p0[v]];
#pragma unroll
        for (int v = 0; v < VEC; ++v) p0[v] = parent[p1[v]];
#pragma unroll
        for (int v = 0; v < VEC; ++v) p1[v] = parent[p0[v]];
        // now p0 = 2 hops above the site's run start, p1 = parent[p0]
#pragma unroll
        for (int v = 0; v < VEC; ++v) { const uint32_t t = p0[v]; p0[v] = p1[v]; p1[v] = t; }
        LabelT out[VEC];
#pragma unroll
        for (int v = 0; v < VEC; ++v) {
            uint32_t root = p0[v];
            if (root != p1[v]) root = sfind(parent, root);
            const uint32_t ry = root / TW, rx = root - ry * TW;
            out[v] = (LabelT)(y0 + ry) * L + (x0 + rx);
        }
        LabelT *dst = labels + (size_t)(y0 + ly) * L + xl;
        if constexpr (sizeof(LabelT) == 4) {
            if constexpr (VEC == 4) *reinterpret_cast<uint4 *>(dst) = make_uint4(out[0], out[1], out[2], out[3]);
            else *reinterpret_cast<uint2 *>(dst) = make_uint2(out[0], out[1]);
        } else {
#pragma unroll
            for (int v = 0; v < VEC; v += 2)
                *reinterpret_cast<ulonglong2 *>(dst + v) = make_ulonglong2(out[v], out[v + 1]);
        }
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
    const uint32_t L = a.L;
    LabelT *labels = reinterpret_cast<LabelT *>(a.labels);
    const uint64_t total = (uint64_t)a.ntiles * (TW + TH);
    for (uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; k < total; k += (uint64_t)gridDim.x * blockDim.x) {
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
            x2 = x; y2 = y + 1 == L ? 0 : y + 1;
            bit = 4 + (x & 3u);
        }
        const size_t i = (size_t)y * L + x;
        if ((a.bonds[i >> 2] >> bit) & 1u) {
            const size_t j = (size_t)y2 * L + x2;
            gunion<LabelT>(labels, gload(labels + i), gload(labels + j));
        }
    }
}

// ---------------------------------------------------------------------------------------------
// k_flip: root of every site (read-only chase; the forest is final after k_merge), coin of the
// root, reflection.  One CTA per TW x TH tile so that the first hop of every chase (the tile-local
// root) is served by L1.  Counts the clusters (#{root == site}).
// ---------------------------------------------------------------------------------------------
template <int VEC, int R, int NW, typename LabelT>
__global__ void __launch_bounds__(NW * 32)
k_flip(const SweepArgs a)
{
    constexpr int TW = 32 * VEC, TH = R * NW;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t L = a.L;
    const LabelT *labels = reinterpret_cast<const LabelT *>(a.labels);
    uint32_t ncl = 0;
    for (uint32_t tile = blockIdx.x; tile < a.ntiles; tile += gridDim.x) {
        const uint32_t ty = tile / a.tiles_x, tx = tile - ty * a.tiles_x;
        const uint32_t xl = tx * TW + lane * VEC;
        const uint32_t yb = ty * TH + warp * R;
        LabelT lab[R][VEC];
        float th[R][VEC];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const size_t i = (size_t)(yb + r) * L + xl;
            if constexpr (sizeof(LabelT) == 4) {
                if constexpr (VEC == 4) {
                    const uint4 v = __ldg(reinterpret_cast<const uint4 *>(labels + i));
                    lab[r][0] = v.x; lab[r][1] = v.y; lab[r][2] = v.z; lab[r][3] = v.w;
                } else {
                    const uint2 v = __ldg(reinterpret_cast<const uint2 *>(labels + i));
                    lab[r][0] = v.x; lab[r][1] = v.y;
                }
            } else {
#pragma unroll
                for (int v = 0; v < VEC; v += 2) {
                    const ulonglong2 q = __ldg(reinterpret_cast<const ulonglong2 *>(labels + i + v));
                    lab[r][v] = q.x; lab[r][v + 1] = q.y;
                }
            }
            load_vec<VEC, false>(a.theta + i, th[r]);
        }
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const size_t i = (size_t)(yb + r) * L + xl;
            LabelT prev_l = (LabelT)~(LabelT)0, prev_root = 0;
            bool prev_coin = false, any = false;
            float out[VEC];
#pragma unroll
            for (int v = 0; v < VEC; ++v) {
                const LabelT l0 = lab[r][v];
                LabelT root;
                bool coin;
                if (v > 0 && l0 == prev_l) {
                    root = prev_root; coin = prev_coin;
                } else {
                    root = l0;
                    if (l0 != (LabelT)(i + v)) {
                        LabelT p = __ldg(labels + root);
                        while (p != root) { root = p; p = __ldg(labels + root); }
                    }
                    coin = (rng(a.seed_lo, a.seed_hi, (uint64_t)root, a.t, TAG_FLIP).x >> 31) != 0u;
                }
                prev_l = l0; prev_root = root; prev_coin = coin;
                ncl += (root == (LabelT)(i + v));
                out[v] = coin ? reflect(th[r][v], a.A) : th[r][v];
                any |= coin;
            }
            if (any) {
                if constexpr (VEC == 4) *reinterpret_cast<float4 *>(a.theta + i) = make_float4(out[0], out[1], out[2], out[3]);
                else *reinterpret_cast<float2 *>(a.theta + i) = make_float2(out[0], out[1]);
            }
        }
    }
    unsigned long long c = warp_sum_u64(ncl);
    __shared__ unsigned long long sc[NW];
    if (lane == 0) sc[warp] = c;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long tot = 0;
        for (int w = 0; w < NW; ++w) tot += sc[w];
        xy_obs *o = a.ring + ((a.t + 1u) % a.ring_cap);
        atomicAdd(reinterpret_cast<unsigned long long *>(&o->n_clusters), tot);
    }
}

// ---------------------------------------------------------------------------------------------
// Small utility kernels (init, export, debug).
// ---------------------------------------------------------------------------------------------
__global__ void k_init_hot(float *theta, uint64_t N, uint32_t seed_lo, uint32_t seed_hi)
{
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (uint64_t)gridDim.x * blockDim.x) {
        const U4 w = rng(seed_lo, seed_hi, i, 0u, TAG_INIT);
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
