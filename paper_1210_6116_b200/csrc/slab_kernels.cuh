// slab_kernels.cuh -- the exchange step of the row-slab sharded sweep (the paper's
// "two-stage process of cluster labeling ... within each GPU and the inter-GPU labeling").
// A rank holds rows [y_off, y_off + rows) of the L x L lattice.  After its local k_bonds / k_label / k_merge:
//   k_slab_edges    the canonical LOCAL root (as an index of the whole lattice) of every site of the slab's first and
//                   last row, and the y-bond bits of the last row: the record every rank contributes to the all-gather.
//   k_stitch_*      replicated on every rank over the gathered records: a union-find over the distinct roots that appear
//                   on the cuts (open-addressing hash table keyed by root, links towards the smaller root, so the root
//                   of a set is the minimum site index of the whole cluster), then for the rank's own edge sites: if
//                   the cluster's canonical root is not the local one, the local root's label entry is overridden with
//                   kSlabSpecial | k and xroot[k] = canonical root (k_flip<..., kSlab> keys the coin by it).
// Product code: shares nothing with oracle/.
#pragma once
#include "xy_kernels.cuh"

namespace xy {

// record of one rank in the gathered buffer: top[L] (u64), bot[L] (u64), ybits[L] (u8, 0/1), padded to 8 bytes
__host__ __device__ inline size_t slab_edge_bytes(uint32_t L) { return (size_t)L * 16 + (((size_t)L + 7) & ~(size_t)7); }

__global__ void k_slab_edges(const uint32_t *labels, const uint8_t *bonds, uint32_t L, uint32_t rows, uint32_t y_off,
                             unsigned char *rec)
{
    uint64_t *top = reinterpret_cast<uint64_t *>(rec), *bot = top + L;
    uint8_t *yb = reinterpret_cast<uint8_t *>(bot + L);
    const uint64_t goff = (uint64_t)y_off * L;
    const uint32_t last = (rows - 1) * L;
    for (uint32_t x = blockIdx.x * blockDim.x + threadIdx.x; x < L; x += gridDim.x * blockDim.x) {
        top[x] = (uint64_t)gfind<uint32_t>(const_cast<uint32_t *>(labels), x) + goff;
        bot[x] = (uint64_t)gfind<uint32_t>(const_cast<uint32_t *>(labels), last + x) + goff;
        yb[x] = (uint8_t)((bonds[(last + x) >> 2] >> (4 + (x & 3u))) & 1u);
    }
}

constexpr uint64_t kHashEmpty = ~0ull;

struct StitchTable {
    uint64_t *key;          // [cap] root (site index in the whole lattice) or kHashEmpty
    uint32_t *parent;       // [cap] slot of the parent (itself for a root)
    uint32_t *slot_of;      // [nranks * 2 L] slot of every gathered edge entry (top entries first, then bot, per rank)
    uint32_t  cap_mask;     // cap - 1 (cap a power of two >= 4 * number of entries)
};

__global__ void k_stitch_clear(StitchTable t)
{
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i <= t.cap_mask; i += gridDim.x * blockDim.x) {
        t.key[i] = kHashEmpty;
        t.parent[i] = i;
    }
}

__device__ __forceinline__ uint32_t stitch_hash(uint64_t k, uint32_t mask)
{
    return (uint32_t)((k * 0x9E3779B97F4A7C15ull) >> 32) & mask;
}

// every gathered top / bot entry gets the slot of its root (inserted on first sight)
__global__ void k_stitch_insert(StitchTable t, const unsigned char *gathered, uint32_t L, uint32_t nranks)
{
    const size_t rb = slab_edge_bytes(L);
    const uint32_t n = nranks * 2u * L;
    for (uint32_t e = blockIdx.x * blockDim.x + threadIdx.x; e < n; e += gridDim.x * blockDim.x) {
        const uint32_t r = e / (2u * L), j = e - r * 2u * L;           // j < L: top[j]; else bot[j - L]
        const uint64_t k = reinterpret_cast<const uint64_t *>(gathered + (size_t)r * rb)[j];
        uint32_t h = stitch_hash(k, t.cap_mask);
        for (;;) {
            const uint64_t old = atomicCAS(reinterpret_cast<unsigned long long *>(t.key + h), (unsigned long long)kHashEmpty,
                                           (unsigned long long)k);
            if (old == kHashEmpty || old == k) break;
            h = (h + 1) & t.cap_mask;
        }
        t.slot_of[e] = h;
    }
}

__device__ __forceinline__ uint32_t stitch_find(const StitchTable &t, uint32_t a)
{
    uint32_t p = *reinterpret_cast<volatile uint32_t *>(t.parent + a);
    while (p != a) { a = p; p = *reinterpret_cast<volatile uint32_t *>(t.parent + a); }
    return a;
}

// the active y bonds of every cut unite the root below rank r's last row with the root above rank r+1's first row
// (the last rank's cut closes the torus)
__global__ void k_stitch_union(StitchTable t, const unsigned char *gathered, uint32_t L, uint32_t nranks)
{
    const size_t rb = slab_edge_bytes(L);
    const uint32_t n = nranks * L;
    for (uint32_t e = blockIdx.x * blockDim.x + threadIdx.x; e < n; e += gridDim.x * blockDim.x) {
        const uint32_t r = e / L, x = e - r * L, r2 = r + 1 == nranks ? 0u : r + 1;
        const uint8_t *yb = gathered + (size_t)r * rb + (size_t)L * 16;
        if (!yb[x]) continue;
        uint32_t a = t.slot_of[r * 2u * L + L + x], b = t.slot_of[r2 * 2u * L + x];
        for (;;) {
            a = stitch_find(t, a);
            b = stitch_find(t, b);
            if (a == b) break;
            // the set's root is the smaller KEY (site index), whatever the slots are
            const uint32_t hi = t.key[a] > t.key[b] ? a : b, lo = hi == a ? b : a;
            if (atomicCAS(t.parent + hi, hi, lo) == hi) break;
            a = hi; b = lo;                                          // hi was linked meanwhile: again from there
        }
    }
}

// my own edge sites: override the local root's label entry where the cluster's canonical root lies elsewhere
__global__ void k_stitch_apply(StitchTable t, const unsigned char *gathered, uint32_t L, uint32_t rank, uint32_t y_off,
                               uint64_t nsites, uint32_t *labels, uint64_t *xroot, unsigned int *bad)
{
    const size_t rb = slab_edge_bytes(L);
    const uint64_t goff = (uint64_t)y_off * L;
    const uint64_t *mine = reinterpret_cast<const uint64_t *>(gathered + (size_t)rank * rb);
    for (uint32_t j = blockIdx.x * blockDim.x + threadIdx.x; j < 2u * L; j += gridDim.x * blockDim.x) {
        const uint64_t k = mine[j];
        if (k - goff >= nsites) { atomicAdd(bad, 1u); continue; }    // not a site of this slab: the record is not this rank's
        if (j != 0 && j != L && mine[j - 1] == k) continue;          // the left neighbour does the same
        const uint32_t root = stitch_find(t, t.slot_of[rank * 2u * L + j]);
        const uint64_t g = t.key[root];
        if (g != k) {
            xroot[j] = g;
            labels[(uint32_t)(k - goff)] = kSlabSpecial | j;         // several edge sites of one local root: same g
        }
    }
}

// label[i] <- canonical label in the whole lattice, as int64 (xy_get_labels of a slab after the stitch)
__global__ void k_slab_labels_to_i64(const uint32_t *labels, const uint64_t *xroot, uint64_t goff, int64_t *out,
                                     uint64_t first, uint64_t n)
{
    for (uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (uint64_t)gridDim.x * blockDim.x) {
        uint32_t r = labels[first + k];
        while (!(r & kSlabSpecial)) {
            const uint32_t p = labels[r];
            if (p == r) break;
            r = p;
        }
        out[k] = (int64_t)((r & kSlabSpecial) ? xroot[r & ~kSlabSpecial] : (uint64_t)r + goff);
    }
}

// PCC on a sharded lattice: the slab's partial sums of one record as 8 doubles (Mx, My, Cx, Sx, Cy, Sy, 0, 0) for the
// all-reduce, and the controller step on the all-reduced sums (replicated on every rank: same inputs, same arithmetic)
__global__ void k_slab_pack_obs(const xy_obs *rec, double *out8)
{
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        out8[0] = rec->Mx; out8[1] = rec->My; out8[2] = rec->Cx; out8[3] = rec->Sx; out8[4] = rec->Cy; out8[5] = rec->Sy;
        out8[6] = 0.0; out8[7] = 0.0;
    }
}

__global__ void k_slab_pcc_feed(DevCtl *c, const double *g8, double N)
{
    if (threadIdx.x == 0 && blockIdx.x == 0) pcc_feed(c, N, g8[2], g8[3], g8[4], g8[5], g8[0], g8[1], 0.0);
}

}  // namespace xy
