// potts_kernels.cuh -- q-state Potts Swendsen-Wang sweep on the labeling core of the XY sweep (
// PAPER.md:30-34 names the authors' Potts / Ising SW codes).  H = -sum_<ij> delta(s_i, s_j), spins one byte per site.
//   k_potts_bonds  (P2, and P5 of the incoming configuration): bond <ij> active iff s_i == s_j and u < 1 - exp(-beta);
//                  the same Philox bond uniforms and the same nibble-packed bond bytes as k_bonds, so that
//                  k_label / k_merge run unchanged.  u < p is an integer compare: u = (w + 0.5) 2^-32 < p
//                  <=> w < T, T = ceil(p 2^32 - 0.5) (host, exact in fp64).  The 16 leading bits of w (call A of
//                  the quad) settle it unless they equal T >> 16; only then call B is drawn.
//   k_potts_flip   (P4): every tile-local root takes the fresh spin of its cluster's canonical label (one Philox
//                  call serves 4 consecutive labels), chasing to the global root if k_merge linked it elsewhere;
//                  every other site copies the spin of its tile root from shared memory.
// Product code: shares nothing with oracle/.
#pragma once
#include "xy_kernels.cuh"

namespace xy {

constexpr uint32_t TAG_POTTS = 5;
constexpr int kPottsMaxQ = 16;

// integer observables and counters of the Potts state (all sums are exact, so plain atomics are reproducible)
struct PottsCtl {
    unsigned long long ex, ey;                 // links with equal spins (incoming state of the last k_potts_bonds)
    unsigned long long count[kPottsMaxQ];      // sites per spin value
    unsigned long long nbx, nby, ncl;          // bonds and clusters of the last sweep
};

struct PottsArgs {
    uint8_t  *spin;
    uint8_t  *bonds;
    PottsCtl *ctl;
    uint32_t  L, q;
    uint32_t  seed_lo, seed_hi, t;
    uint64_t  T;                               // threshold: bond iff equal spins and w < T (0 .. 2^32)
};

__device__ __forceinline__ uint32_t eq4_bits(uint32_t a, uint32_t b)   // bit j = byte j of a equals byte j of b
{
    // spins are below 128: the low 7 bits of a byte of a ^ b are zero iff the bytes are equal, and adding 0x7f then
    // leaves bit 7 clear exactly there (no carry crosses a byte)
    const uint32_t m = ~((a ^ b) + 0x7f7f7f7fu) & 0x80808080u;
    return (m >> 7 | m >> 14 | m >> 21 | m >> 28) & 15u;
}

// kBonds = false: observables only (xy_potts_measure of a state no sweep has looked at yet).  KQ: number of spin
// values counted (q <= KQ; 4, 8 or 16).  A thread owns quads of 4 consecutive sites (one bond byte, one Philox call).
template <bool kBonds, int KQ>
__global__ void __launch_bounds__(256)
k_potts_bonds(const PottsArgs a)
{
    const uint32_t L = a.L, q = a.q;
    const uint32_t nquads = (uint32_t)(((uint64_t)L * L) >> 2), qpr = L >> 2;      // quads in all, per row
    const uint32_t Th = (uint32_t)(a.T >> 16), Tl = (uint32_t)(a.T & 0xffffu);
    unsigned long long ex = 0, ey = 0, nbx = 0, nby = 0;
    uint32_t cnt[KQ];
#pragma unroll
    for (int k = 0; k < KQ; ++k) cnt[k] = 0;

    for (uint32_t qd = blockIdx.x * blockDim.x + threadIdx.x; qd < nquads; qd += gridDim.x * blockDim.x) {
        const uint64_t i0 = (uint64_t)qd << 2;
        const uint32_t y = qd / qpr, x = (qd - y * qpr) << 2;
        const uint32_t own = __ldg(reinterpret_cast<const uint32_t *>(a.spin + i0));
        const uint32_t xr = x + 4 == L ? 0u : x + 4;
        const uint32_t nb = __ldg(a.spin + (uint64_t)y * L + xr);
        const uint32_t yd = y + 1 == L ? 0u : y + 1;
        const uint32_t down = __ldg(reinterpret_cast<const uint32_t *>(a.spin + (uint64_t)yd * L + x));
        const uint32_t eqx = eq4_bits(own, (own >> 8) | (nb << 24));
        const uint32_t eqy = eq4_bits(own, down);
        ex += __popc(eqx);
        ey += __popc(eqy);
        if constexpr (KQ == 4) {                     // two bits per spin: four masks from two bit planes
            const uint32_t b0 = own & 0x01010101u, b1 = (own >> 1) & 0x01010101u;
            cnt[3] += __popc(b0 & b1);
            cnt[1] += __popc(b0 & ~b1);
            cnt[2] += __popc(b1 & ~b0);
            cnt[0] += __popc(0x01010101u & ~(b0 | b1));
        } else {
#pragma unroll
            for (int k = 0; k < KQ; ++k) cnt[k] += __popc(eq4_bits(own, 0x01010101u * (uint32_t)k));
        }
        if constexpr (kBonds) {
            const U4 wA = rng(a.seed_lo, a.seed_hi, qd, a.t, TAG_BOND);
            const uint32_t w[4] = {wA.x, wA.y, wA.z, wA.w};
            // h < Th as the sign of h - Th (both below 2^17), shifted into place by funnel shifts
            uint32_t xn = 0, yn = 0;
            bool tie = false;
#pragma unroll
            for (int j = 3; j >= 0; --j) {
                const uint32_t dx = (w[j] & 0xffffu) - Th, dy = (w[j] >> 16) - Th;
                xn = __funnelshift_l(dx, xn, 1);
                yn = __funnelshift_l(dy, yn, 1);
                tie = tie || dx == 0u || dy == 0u;
            }
            if (tie) {                                     // rare (2^-16 per decision): the trailing 16 bits decide
                const U4 wB = rng(a.seed_lo, a.seed_hi, qd, a.t, TAG_BOND_LO);
                const uint32_t v[4] = {wB.x, wB.y, wB.z, wB.w};
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    if ((w[j] & 0xffffu) == Th) xn |= ((v[j] & 0xffffu) < Tl ? 1u : 0u) << j;
                    if ((w[j] >> 16) == Th) yn |= ((v[j] >> 16) < Tl ? 1u : 0u) << j;
                }
            }
            xn &= eqx;
            yn &= eqy;
            nbx += __popc(xn);
            nby += __popc(yn);
            a.bonds[qd] = (uint8_t)(xn | (yn << 4));
        }
    }
    ex = warp_sum_u64(ex); ey = warp_sum_u64(ey);
    nbx = warp_sum_u64(nbx); nby = warp_sum_u64(nby);
    unsigned long long c64[KQ];
#pragma unroll
    for (int k = 0; k < KQ; ++k) c64[k] = warp_sum_u64(cnt[k]);
    if ((threadIdx.x & 31) == 0) {
        atomicAdd(&a.ctl->ex, ex);
        atomicAdd(&a.ctl->ey, ey);
#pragma unroll
        for (int k = 0; k < KQ; ++k)
            if (k < (int)q && c64[k]) atomicAdd(&a.ctl->count[k], c64[k]);
        if constexpr (kBonds) {
            atomicAdd(&a.ctl->nbx, nbx);
            atomicAdd(&a.ctl->nby, nby);
        }
    }
}

__device__ __forceinline__ uint32_t potts_draw(uint32_t seed_lo, uint32_t seed_hi, uint64_t rho, uint32_t t, uint32_t q)
{
    const U4 c = rng(seed_lo, seed_hi, rho >> 2, t, TAG_POTTS);
    const uint32_t sel = (uint32_t)rho & 3u;
    const uint32_t w = sel == 0 ? c.x : sel == 1 ? c.y : sel == 2 ? c.z : c.w;
    return __umulhi(w, q);                                              // floor(q w / 2^32)
}

// One CTA per TW x TH tile (the tiles of k_label), 4 consecutive sites x TH/RPP rows per thread.
template <int WPR, int TH, typename LabelT>
__global__ void __launch_bounds__(WPR * TH)
k_potts_flip(const SweepArgs a, const PottsArgs p)
{
    constexpr int TW = 32 * WPR, NT = WPR * TH;
    constexpr int Q = TW / 4, RPP = NT / Q, NP = TH / RPP;
    __shared__ uint8_t fresh[TW * TH];               // fresh spin of the tile root at tile-local index loc
    __shared__ uint16_t queue[TW * TH];              // tile-local indices of the tile roots
    __shared__ uint32_t nqueue;
    __shared__ unsigned long long sc[NT / 32];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t L = a.L;
    const LabelT *labels = reinterpret_cast<const LabelT *>(a.labels);
    const uint32_t tile = blockIdx.x;
    const uint32_t ty = tile / a.tiles_x, tx = tile - ty * a.tiles_x;
    const uint32_t x0 = tx * TW, y0 = ty * TH;
    const int q4 = tid % Q, rq = tid / Q;
    const LabelT gbase = (LabelT)y0 * L + x0;

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

    // ---- tile roots are queued (a tile has TW*TH of them at most), then draw densely: their own label if it still
    //      is a global root, else the root k_merge linked them to ----
    if (tid == 0) nqueue = 0;
    __syncthreads();
    uint32_t rb = 0, merged = 0, ncl = 0;             // root bits of my sites; of those, the ones k_merge linked elsewhere
#pragma unroll
    for (int k = 0; k < NP; ++k) {
        const size_t i = (size_t)(y0 + k * RPP + rq) * L + x0 + 4 * q4;
        LabelT lab[4];
        load_labels(i, lab);                         // coalesced; read again (from L2) in the last phase
        rb |= ((__ldg(reinterpret_cast<const uint8_t *>(a.rootmask) + (i >> 3)) >> (i & 4u)) & 15u) << (4 * k);
#pragma unroll
        for (int v = 0; v < 4; ++v)
            if (lab[v] != (LabelT)(i + v)) merged |= 1u << (4 * k + v);
    }
    merged &= rb;
    {
        // one slot reservation per warp: ballots of the four-bit counts
        const uint32_t n = __popc(rb);
        uint32_t pre = n;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t t = __shfl_up_sync(0xffffffffu, pre, o);
            if (lane >= o) pre += t;
        }
        uint32_t wbase = 0;
        if (lane == 31) wbase = atomicAdd(&nqueue, pre);
        wbase = __shfl_sync(0xffffffffu, wbase, 31);
        uint32_t slot = wbase + pre - n, bits = rb;
        while (bits) {
            const int b = __ffs(bits) - 1;
            bits &= bits - 1;
            // tile-local index (< 2^15) and, in bit 15, whether the root was linked elsewhere
            queue[slot++] = (uint16_t)((((b >> 2) * RPP + rq) * TW + 4 * q4 + (b & 3)) | (((merged >> b) & 1u) << 15));
        }
    }
    __syncthreads();
    for (uint32_t j = tid; j < nqueue; j += NT) {
        const uint32_t e = queue[j], loc = e & 0x7fffu;
        const LabelT self = gbase + (LabelT)(loc / TW) * L + (loc % TW);
        LabelT root = self;
        if (!(e & 0x8000u)) {
            ++ncl;
        } else {                                                         // read-only chase: the forest is final
            root = __ldg(labels + self);
            LabelT up = __ldg(labels + root);
            while (up != root) { XY_CHECK(CHK_GLABEL, up < root); root = up; up = __ldg(labels + root); }
        }
        fresh[loc] = (uint8_t)potts_draw(p.seed_lo, p.seed_hi, (uint64_t)root, p.t, p.q);
    }
    __syncthreads();

    // ---- every site takes the fresh spin of its tile root ----
    const uint32_t Lm = L - TW;
#pragma unroll
    for (int k = 0; k < NP; ++k) {
        const int row = k * RPP + rq;
        const uint32_t loc0 = row * TW + 4 * q4;
        const size_t i = (size_t)(y0 + row) * L + x0 + 4 * q4;
        LabelT lab[4];
        load_labels(i, lab);
        uint32_t out = 0;
#pragma unroll
        for (int v = 0; v < 4; ++v) {
            const uint32_t d = (uint32_t)(lab[v] - gbase);              // r*L + c, < TH*L <= 2^22
            const uint32_t rr = __umulhi(d, a.Ldiv_mul) >> a.Ldiv_shift;
            const uint32_t loc = ((rb >> (4 * k + v)) & 1u) ? loc0 + v : d - rr * Lm;
            XY_CHECK(CHK_LOC, loc < (uint32_t)(TW * TH));
            out |= (uint32_t)fresh[loc] << (8 * v);
        }
        *reinterpret_cast<uint32_t *>(p.spin + i) = out;
    }

    unsigned long long c = warp_sum_u64(ncl);
    if (lane == 0) sc[warp] = c;
    __syncthreads();
    if (tid == 0) {
        unsigned long long tot = 0;
        for (int w = 0; w < NT / 32; ++w) tot += sc[w];
        atomicAdd(&p.ctl->ncl, tot);
    }
}

__global__ void k_potts_init_hot(uint8_t *spin, uint64_t N, uint32_t q, uint32_t seed_lo, uint32_t seed_hi)
{
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (uint64_t)gridDim.x * blockDim.x) {
        const U4 w = rng(seed_lo, seed_hi, i, 0u, TAG_INIT);
        spin[i] = (uint8_t)__umulhi(w.x, q);
    }
}

__global__ void k_potts_check_spins(const uint8_t *spin, uint64_t N, uint32_t q, unsigned int *flag)
{
    bool bad = false;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (uint64_t)gridDim.x * blockDim.x)
        bad |= spin[i] >= q;
    if (bad) atomicOr(flag, 1u);
}

}  // namespace xy
