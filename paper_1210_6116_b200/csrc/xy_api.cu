// xy_api.cu -- C-ABI boundary (include/xy.h) of the B200-native XY Swendsen-Wang sweep.
// Host logic only: argument checks, workspace carving, per-sweep scalar parameters (direction
// phi_t from the host-side Philox, the reflection constant), launch sequencing, ring bookkeeping.
// Every step of the hot path runs in the kernels of xy_kernels.cuh; there is no CPU fallback.
#include "xy_kernels.cuh"
#include "slab_kernels.cuh"

#include <curand_philox4x32_x.h>   // NVIDIA's curand_Philox4x32_10, for xy_debug_curand_philox only

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <mutex>
#include <new>
#include <utility>
#include <vector>

using namespace xy;

namespace {

thread_local char g_err[512] = "";

int fail(int code, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
    return code;
}

#define CUDA_TRY(expr)                                                                       \
    do {                                                                                     \
        cudaError_t e_ = (expr);                                                             \
        if (e_ != cudaSuccess)                                                               \
            return fail(e_ == cudaErrorMemoryAllocation ? XY_ERR_NOMEM : XY_ERR_CUDA,        \
                        "%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e_), __FILE__, __LINE__); \
    } while (0)

constexpr uint32_t kRingCap = 16384;       // per-sweep records kept on the device
constexpr uint32_t kMaxGrid = 148 * 16;    // upper bound for the persistent grids (partials array)
constexpr size_t kStageBytes = 64u << 20;  // staging buffer of the debug getters

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

struct Layout {
    size_t theta, labels, bonds, rootmask, partials, ring, fring, ctl, tab, edges, xroot, pccbuf, stitch, total;
};

// stitch table of a slab for nranks slabs: cap hash slots (key u64 + parent u32) and one slot index per gathered edge entry
uint32_t stitch_cap(uint64_t entries)
{
    uint32_t cap = 1024;
    while (cap < 4 * entries) cap <<= 1;
    return cap;
}
size_t stitch_bytes(uint32_t L, uint32_t nranks)
{
    const uint64_t entries = (uint64_t)nranks * 2u * L;
    return (size_t)stitch_cap(entries) * 12 + entries * 4;
}
// number of equal slabs the lattice splits into when every rank holds `rows` rows: the stitch table inside the workspace is
// sized for it (another nranks at xy_slab_flip still works: that table is then allocated apart)
uint32_t default_ranks(uint32_t L, uint32_t rows) { return (L + rows - 1) / rows; }

// rows == L and slab == false: a whole lattice.  A slab holds `rows` rows plus one halo row of
// theta, its edge record for the all-gather and the table of overridden roots.
Layout make_layout(uint32_t L, uint32_t flags, uint32_t rows = 0, bool slab = false)
{
    if (rows == 0) rows = L;
    const size_t N = (size_t)rows * L;
    const size_t lw = (flags & XY_FLAG_LABELS64) ? 8 : 4;
    Layout o;
    size_t off = 0;
    o.theta = off;    off = align_up(off + (N + (slab ? L : 0)) * 4, 256);
    o.labels = off;   off = align_up(off + N * lw, 256);
    o.bonds = off;    off = align_up(off + N / 4, 256);
    o.rootmask = off; off = align_up(off + N / 8, 256);
    o.partials = off; off = align_up(off + (size_t)kMaxGrid * kPartialStride * 8, 256);
    o.ring = off;     off = align_up(off + (size_t)kRingCap * sizeof(xy_obs), 256);
    o.fring = off;    off = align_up(off + ((flags & XY_FLAG_FOURIER) ? (size_t)kRingCap * sizeof(xy_fourier) : 0), 256);
    o.ctl = off;      off = align_up(off + sizeof(DevCtl), 256);
    o.tab = off;      off = align_up(off + (size_t)(kTabN + 1) * sizeof(double2), 256);
    o.edges = off;    off = align_up(off + (slab ? slab_edge_bytes(L) : 0), 256);
    o.xroot = off;    off = align_up(off + (slab ? (size_t)2 * L * 8 : 0), 256);
    o.pccbuf = off;   off = align_up(off + (slab ? (size_t)16 * 8 : 0), 256);
    o.stitch = off;   off = align_up(off + (slab ? stitch_bytes(L, default_ranks(L, rows)) : 0), 256);
    o.total = off;
    return o;
}

// The four kernels of a sweep are launched with programmatic stream serialization (xy_device.cuh, pdl_wait): the next
// kernel's CTAs may become resident and run their prologue while the previous grid drains.  XY_NO_PDL=1 in the
// environment launches them the plain way, XY_PDL_MASK=<bits> only the named kernels with the attribute (A/B runs).
enum { PDL_BONDS = 1, PDL_LABEL = 2, PDL_MERGE = 4, PDL_FLIP = 8 };
int pdl_mask()
{
    static const int mask = [] {
        if (const char *e = getenv("XY_NO_PDL")) if (e[0] == '1') return 0;
        if (const char *e = getenv("XY_PDL_MASK")) return atoi(e) & 15;
        return 15;
    }();
    return mask;
}

template <typename... KArgs, typename... Args>
cudaError_t launch_chain(int which, void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args &&...args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = (pdl_mask() & which) ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, std::forward<Args>(args)...);
}

// One set of launchers per (tile geometry, label width).
struct Kernels {
    // what: 0 = sweep with observables, 1 = observables only, 2 = sweep without observables
    cudaError_t (*bonds)(const SweepArgs &, int what, bool fourier, int grid, cudaStream_t);
    void (*label)(const SweepArgs &, cudaStream_t);
    void (*merge)(const SweepArgs &, cudaStream_t);
    void (*flip)(const SweepArgs &, int grid, cudaStream_t);
    void (*flip_slab)(const SweepArgs &, cudaStream_t);
    int (*prepare)(bool fourier, int *bonds_obs, int *bonds_noobs, int *fl);
    int tw, th, rs;
};

// rows per warp strip in k_bonds: 32 (1/32 halo recompute) on large lattices; 8 where 32-row strips would
// leave warps without work or with one long serial strip (L <= 4096: fewer than 2 strips per resident warp)
constexpr int kRSLarge = 32, kRSSmall = 8;

template <int VEC, int R, int NW, int RS, typename LabelT>
struct KS {
    template <bool kB, bool kO, bool kF>
    static cudaError_t bonds_launch(const SweepArgs &a, int grid, cudaStream_t st)
    {
        return launch_chain(PDL_BONDS, k_bonds<VEC, RS, kB, kO, kF>, grid, BondsShape<kO>::warps * 32, k_bonds_smem_bytes<kO>(), st, a);
    }
    template <bool kB, bool kO>
    static cudaError_t bonds_slab_launch(const SweepArgs &a, int grid, cudaStream_t st)
    {
        return launch_chain(PDL_BONDS, k_bonds<VEC, RS, kB, kO, false, true>, grid, BondsShape<kO>::warps * 32, k_bonds_smem_bytes<kO>(), st, a);
    }
    static cudaError_t bonds(const SweepArgs &a, int what, bool fourier, int grid, cudaStream_t st)
    {
        if (a.open_y) {
            if (what == 2) return bonds_slab_launch<true, false>(a, grid, st);
            return what == 1 ? bonds_slab_launch<false, true>(a, grid, st) : bonds_slab_launch<true, true>(a, grid, st);
        }
        if (what == 2) return bonds_launch<true, false, false>(a, grid, st);
        if (fourier) return what == 1 ? bonds_launch<false, true, true>(a, grid, st) : bonds_launch<true, true, true>(a, grid, st);
        return what == 1 ? bonds_launch<false, true, false>(a, grid, st) : bonds_launch<true, true, false>(a, grid, st);
    }
    static void label(const SweepArgs &a, cudaStream_t st)
    {
        launch_chain(PDL_LABEL, k_label<VEC, R * NW, LabelT>, a.ntiles, VEC * R * NW, k_label_smem_bytes<VEC, R * NW>(), st, a);
    }
    static void merge(const SweepArgs &a, cudaStream_t st)
    {
        const uint64_t total = (uint64_t)a.ntiles * (32 * VEC + R * NW);
        uint64_t blocks = (total + 255) / 256;
        if (blocks > 148ull * 64) blocks = 148ull * 64;
        // measured (profiles/r3_pdl.md): above L = 4096 an early-resident k_merge costs more than its launch gap saves
        launch_chain(a.L <= 4096 ? PDL_MERGE : 0, k_merge<32 * VEC, R * NW, LabelT>, (unsigned)blocks, 256, 0, st, a);
    }
    static void flip(const SweepArgs &a, int grid, cudaStream_t st)
    {
        (void)grid;
        launch_chain(PDL_FLIP, k_flip<VEC, R * NW, LabelT>, a.ntiles, VEC * R * NW, 0, st, a);
    }
    static void flip_slab(const SweepArgs &a, cudaStream_t st)
    {
        if constexpr (sizeof(LabelT) == 4) launch_chain(PDL_FLIP, k_flip<VEC, R * NW, LabelT, true>, a.ntiles, VEC * R * NW, 0, st, a);
    }
    template <bool kB, bool kO, bool kF>
    static cudaError_t bonds_prepare(int *occ)
    {
        // opt in to more than 48 KB of dynamic shared memory: per device, so set at every state creation
        cudaError_t e = cudaFuncSetAttribute(k_bonds<VEC, RS, kB, kO, kF>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)k_bonds_smem_bytes<kO>());
        if (e != cudaSuccess) return e;
        int n = 0;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k_bonds<VEC, RS, kB, kO, kF>, BondsShape<kO>::warps * 32,
                                                          k_bonds_smem_bytes<kO>());
        if (occ && (*occ == 0 || n < *occ)) *occ = n;
        return e;
    }
    // sets the kernel attributes on the current device; CTAs per SM of the k_bonds variants with observables
    // (they share ONE grid so that their fixed-order sums agree bitwise), of the variant without, of k_flip
    static int prepare(bool fourier, int *bonds_obs, int *bonds_noobs, int *fl)
    {
        cudaError_t e;
        *bonds_obs = 0; *bonds_noobs = 0;
        if (fourier) {
            e = bonds_prepare<true, true, true>(bonds_obs);
            if (e == cudaSuccess) e = bonds_prepare<false, true, true>(bonds_obs);
        } else {
            e = bonds_prepare<true, true, false>(bonds_obs);
            if (e == cudaSuccess) e = bonds_prepare<false, true, false>(bonds_obs);
        }
        if (e == cudaSuccess) e = bonds_prepare<true, false, false>(bonds_noobs);
        // the slab variants: same shapes and shared memory
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_bonds<VEC, RS, true, true, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)k_bonds_smem_bytes<true>());
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_bonds<VEC, RS, false, true, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)k_bonds_smem_bytes<true>());
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_bonds<VEC, RS, true, false, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)k_bonds_smem_bytes<false>());
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(k_label<VEC, R * NW, LabelT>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                     (int)k_label_smem_bytes<VEC, R * NW>());
        if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(fl, k_flip<VEC, R * NW, LabelT>, VEC * R * NW, 0);
        return (int)e;
    }
    static Kernels get()
    {
        return Kernels{&bonds, &label, &merge, &flip, &flip_slab, &prepare, 32 * VEC, R * NW, RS};
    }
};

constexpr int kR = 4, kNW = 8;   // label / flip tiles: TH = kR * kNW = 32 rows; 128 x 32 (VEC 4) or 64 x 32 (VEC 2)

Kernels pick_kernels(uint32_t L, bool l64)
{
    const bool small = L <= 4096;
    if (L % 128 == 0) {
        if (small) return l64 ? KS<4, kR, kNW, kRSSmall, uint64_t>::get() : KS<4, kR, kNW, kRSSmall, uint32_t>::get();
        return l64 ? KS<4, kR, kNW, kRSLarge, uint64_t>::get() : KS<4, kR, kNW, kRSLarge, uint32_t>::get();
    }
    if (small) return l64 ? KS<2, kR, kNW, kRSSmall, uint64_t>::get() : KS<2, kR, kNW, kRSSmall, uint32_t>::get();
    return l64 ? KS<2, kR, kNW, kRSLarge, uint64_t>::get() : KS<2, kR, kNW, kRSLarge, uint32_t>::get();
}

__global__ void k_debug_curand_philox(const uint32_t *ctr, const uint32_t *key, uint32_t *out, size_t n)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const uint4 c = make_uint4(ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3]);
    const uint2 k = make_uint2(key[2 * i], key[2 * i + 1]);
    const uint4 w = curand_Philox4x32_10(c, k);
    out[4 * i] = w.x; out[4 * i + 1] = w.y; out[4 * i + 2] = w.z; out[4 * i + 3] = w.w;
}

__global__ void k_ctl_init(DevCtl *c, xy_obs *ring, uint32_t ring_cap, uint64_t T)
{
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        memset(c, 0, sizeof(DevCtl));
        xy_obs *o = ring + (T % ring_cap);
        memset(o, 0, sizeof(xy_obs));
        o->sweep = T;
        const double qnan = __longlong_as_double(0x7ff8000000000000LL);
        o->beta = qnan;
        o->E = qnan; o->Mx = qnan; o->My = qnan; o->Cx = qnan; o->Sx = qnan; o->Cy = qnan; o->Sy = qnan;
    }
}

__global__ void k_ring_reset(xy_obs *ring, uint32_t ring_cap, uint64_t T)
{
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        xy_obs *o = ring + (T % ring_cap);
        memset(o, 0, sizeof(xy_obs));
        o->sweep = T;
        const double qnan = __longlong_as_double(0x7ff8000000000000LL);
        o->beta = qnan;
        o->E = qnan; o->Mx = qnan; o->My = qnan; o->Cx = qnan; o->Sx = qnan; o->Cy = qnan; o->Sy = qnan;
    }
}

__global__ void k_check_angles(const float *theta, uint64_t N, unsigned int *flag)
{
    bool bad = false;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (uint64_t)gridDim.x * blockDim.x) {
        const float v = theta[i];
        bad |= !(v >= 0.0f && v <= 6.2831855f);
    }
    if (bad) atomicOr(flag, 1u);
}

struct PccSetup {
    double beta0, dbeta0;
    unsigned long long halve_every;
    double dbeta_min, target;
    unsigned int window, dirs;
    double *trace_beta, *trace_bY;
    unsigned long long trace_cap;
};

// fresh: a new run (controller reset); else the controller continues from its state (xy_pcc_continue), only the
// schedule and the trace arrays of this call are set
__global__ void k_pcc_setup(DevCtl *c, PccSetup s, int fresh)
{
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        if (fresh) {
            c->beta = s.beta0; c->dbeta = s.dbeta0;
            c->acc_e = 0; c->acc_s2 = 0; c->k = 0; c->n_dec = 0;
            c->stage_sum = 0; c->last_sum = 0; c->stage_cnt = 0; c->last_cnt = 0;
            c->sum_m2 = 0; c->sum_chik = 0; c->n_acc = 0;
        }
        c->trace_base = c->n_dec;
        c->halve_every = s.halve_every; c->dbeta_min = s.dbeta_min; c->target = s.target;
        c->window = s.window; c->dirs = s.dirs;
        c->trace_beta = s.trace_beta; c->trace_bY = s.trace_bY; c->trace_cap = s.trace_cap;
    }
}

}  // namespace

struct xy_state {
    uint32_t L = 0, flags = 0;
    uint32_t rows = 0, y_off = 0;   // the state holds rows [y_off, y_off + rows) of the L x L lattice (rows == L: all of it)
    bool slab = false;              // created by xy_slab_create: open in y, halo row, stitch
    bool slab_labelled = false;     // xy_slab_label done, xy_slab_flip pending
    StitchTable stitch{};           // replicated union-find over the cut roots: inside the workspace for L / rows slabs,
    uint32_t stitch_ranks = 0;      //   allocated apart (stitch_owned) if xy_slab_flip is called with another nranks
    bool stitch_owned = false;
    SweepArgs pending{};            // arguments of the sweep between xy_slab_label and xy_slab_flip
    uint64_t N = 0, seed = 0;       // N: sites held by this state
    uint64_t T = 0;                 // sweeps done
    int device = 0;
    bool owns_ws = false;
    char *ws = nullptr;
    Layout lay{};
    Kernels ker{};
    int grid_bonds = 0, grid_bonds_noobs = 0, grid_fl = 0;
    int obs_mode = XY_OBS_ALL;      // xy_set_obs_mode
    cudaStream_t stream = nullptr;
    bool have_sweep = false;        // bonds / labels of a sweep exist
    bool labels_flat = false;
    uint64_t obs_valid_T = UINT64_MAX;   // ring record whose observables are (or will be, in stream order) filled
    uint64_t oldest_T = 0;          // oldest record still meaningful in the ring
    bool fix_phi = false;
    double phi_fixed = 0.0;
    void *stage = nullptr;          // lazily allocated device staging for the getters
    uint64_t launches = 0;          // kernels launched so far
    // per-kernel timing (xy_debug_kernel_timing)
    bool timing = false;
    std::vector<cudaEvent_t> ev;    // 4 events per timed sweep
    size_t ev_used = 0;
    double t_ms[4] = {0, 0, 0, 0};
    uint64_t t_n[4] = {0, 0, 0, 0};

    float *theta() const { return reinterpret_cast<float *>(ws + lay.theta); }
    void *labels() const { return ws + lay.labels; }
    uint8_t *bonds() const { return reinterpret_cast<uint8_t *>(ws + lay.bonds); }
    uint32_t *rootmask() const { return reinterpret_cast<uint32_t *>(ws + lay.rootmask); }
    double *partials() const { return reinterpret_cast<double *>(ws + lay.partials); }
    xy_obs *ring() const { return reinterpret_cast<xy_obs *>(ws + lay.ring); }
    DevCtl *ctl() const { return reinterpret_cast<DevCtl *>(ws + lay.ctl); }
    double2 *tab() const { return reinterpret_cast<double2 *>(ws + lay.tab); }
    unsigned char *edges() const { return reinterpret_cast<unsigned char *>(ws + lay.edges); }
    uint64_t *xroot() const { return reinterpret_cast<uint64_t *>(ws + lay.xroot); }
    double *pccbuf() const { return reinterpret_cast<double *>(ws + lay.pccbuf); }   // [0..7] partial, [8..15] all-reduced
    bool l64() const { return (flags & XY_FLAG_LABELS64) != 0; }
    bool fourier() const { return (flags & XY_FLAG_FOURIER) != 0; }
    xy_fourier *fring() const { return reinterpret_cast<xy_fourier *>(ws + lay.fring); }
};

namespace {

struct DeviceGuard {
    int prev = -1;
    explicit DeviceGuard(int dev) { cudaGetDevice(&prev); if (prev != dev) cudaSetDevice(dev); else prev = -1; }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

void set_stitch(xy_state *s, void *p, uint32_t nranks)
{
    const uint32_t cap = stitch_cap((uint64_t)nranks * 2u * s->L);
    s->stitch.key = static_cast<uint64_t *>(p);
    s->stitch.parent = reinterpret_cast<uint32_t *>(s->stitch.key + cap);
    s->stitch.slot_of = s->stitch.parent + cap;
    s->stitch.cap_mask = cap - 1;
    s->stitch_ranks = nranks;
}

int check_L(uint32_t L)
{
    if (L < 64 || L > 65536 || (L % 64) != 0)
        return fail(XY_ERR_UNSUPPORTED_L, "L=%u unsupported: need a multiple of 64 in [64, 65536]", L);
    return XY_OK;
}

// d / L for d < 2^22 (k_flip): with 2^sh <= L < 2^(sh+1), M = ceil(2^(31+sh) / L) <= 2^31 and
// floor(d M / 2^(31+sh)) = floor(d / L) because the excess d e / 2^(31+sh) < 2^(-9-sh) < 1/L
void set_Ldiv(SweepArgs &a, uint32_t L)
{
    uint32_t sh = 0;
    while ((2u << sh) <= L) ++sh;
    const uint64_t num = 1ull << (31 + sh);
    a.Ldiv_mul = (uint32_t)((num + L - 1) / L);
    a.Ldiv_shift = sh - 1;
}

SweepArgs base_args(const xy_state *s)
{
    SweepArgs a;
    memset(&a, 0, sizeof a);
    a.theta = s->theta();
    a.labels = s->labels();
    a.bonds = s->bonds();
    a.rootmask = s->rootmask();
    a.partials = s->partials();
    a.ctl = s->ctl();
    a.ring = s->ring();
    a.ring_cap = kRingCap;
    a.L = s->L;
    a.tiles_x = s->L / s->ker.tw;
    a.ntiles = a.tiles_x * (s->rows / s->ker.th);
    a.rows = s->rows;
    a.y_off = s->y_off;
    a.open_y = s->slab ? 1 : 0;
    a.xroot = s->xroot();
    set_Ldiv(a, s->L);
    a.seed_lo = (uint32_t)(s->seed & 0xffffffffu);
    a.seed_hi = (uint32_t)(s->seed >> 32);
    for (uint32_t r = 0; r < 10; ++r) {
        a.rk[2 * r] = a.seed_lo + r * 0x9E3779B9u;
        a.rk[2 * r + 1] = a.seed_hi + r * 0xBB67AE85u;
    }
    a.t = (uint32_t)s->T;
    a.cphi = 1.0;                   // observables-only launches use the unrotated frame (phi = 0)
    a.sincos_tab = s->tab();
    a.fring = s->fourier() ? s->fring() : nullptr;
    {
        const long double ang = 6.283185307179586476925286766559L / (long double)s->L;
        a.ck1 = (double)cosl(ang);
        a.sk1 = (double)sinl(ang);
    }
    return a;
}

// direction of sweep t and the constants derived from it (host side, once per sweep)
void set_direction(const xy_state *s, uint64_t t, SweepArgs &a)
{
    double phi;
    if (s->fix_phi) {
        phi = s->phi_fixed;
    } else {
        const U4 w = rng((uint32_t)(s->seed & 0xffffffffu), (uint32_t)(s->seed >> 32), 0, (uint32_t)t, TAG_DIR);
        phi = kTwoPi * ((double)w.x * (1.0 / 4294967296.0));
    }
    a.phi = phi;
    a.cphi = std::cos(phi);
    a.sphi = std::sin(phi);
    volatile double A = 2.0 * phi;       // volatile: no contraction of the multiply-add on the host
    A = A + kPi;
    while (A >= kTwoPi) A = A - kTwoPi;
    a.A = A;
}

int ensure_stage(xy_state *s)
{
    if (!s->stage) CUDA_TRY(cudaMalloc(&s->stage, kStageBytes));
    return XY_OK;
}

// enqueue the observables of the current configuration (record T) if they are not on their way
int ensure_obs(xy_state *s, int feed_pcc)
{
    if (s->obs_valid_T == s->T && !feed_pcc) return XY_OK;
    SweepArgs a = base_args(s);
    a.obs_fill = 1;
    a.feed_pcc = feed_pcc;
    CUDA_TRY(s->ker.bonds(a, 1, s->fourier(), s->grid_bonds, s->stream));
    s->launches += 1;
    s->obs_valid_T = s->T;
    return XY_OK;
}

// slab: did an earlier xy_slab_flip meet edge records that were not this rank's (k_stitch_apply skipped them)?  Blocking.
int slab_stitch_check(xy_state *s)
{
    if (!s->slab) return XY_OK;
    unsigned int bad = 0;
    CUDA_TRY(cudaMemcpyAsync(&bad, &s->ctl()->stitch_bad, sizeof bad, cudaMemcpyDeviceToHost, s->stream));
    CUDA_TRY(cudaStreamSynchronize(s->stream));
    if (!bad) return XY_OK;
    CUDA_TRY(cudaMemsetAsync(&s->ctl()->stitch_bad, 0, sizeof bad, s->stream));
    return fail(XY_ERR_ARG, "xy_slab_flip: %u edge sites of the gathered record of this rank lie outside the slab "
                            "(wrong rank or nranks, or records not in rank order); the labels of that sweep are not valid", bad);
}

constexpr size_t kTimedSweepsPerFlush = 1024;
constexpr int kTimedKernels = 4;      // k_bonds, k_label, k_merge, k_flip

int timing_flush(xy_state *s)
{
    if (s->ev_used == 0) return XY_OK;
    CUDA_TRY(cudaEventSynchronize(s->ev[s->ev_used - 1]));
    for (size_t k = 0; k + kTimedKernels + 1 <= s->ev_used; k += kTimedKernels + 1) {
        for (int j = 0; j < kTimedKernels; ++j) {
            float ms = 0;
            CUDA_TRY(cudaEventElapsedTime(&ms, s->ev[k + j], s->ev[k + j + 1]));
            s->t_ms[j] += ms;
            s->t_n[j] += 1;
        }
    }
    s->ev_used = 0;
    return XY_OK;
}

int timing_mark(xy_state *s)
{
    if (s->ev_used == s->ev.size()) {
        cudaEvent_t e;
        CUDA_TRY(cudaEventCreate(&e));
        s->ev.push_back(e);
    }
    CUDA_TRY(cudaEventRecord(s->ev[s->ev_used++], s->stream));
    return XY_OK;
}

// one sweep at the state's counter; beta_from_ctl: PCC mode
int enqueue_sweep(xy_state *s, double beta, int beta_from_ctl, int feed_pcc)
{
    if (s->T >= 0xffffffffull) return fail(XY_ERR_STATE, "sweep counter would reach 2^32");
    SweepArgs a = base_args(s);
    set_direction(s, s->T, a);
    a.beta = beta;
    a.beta_from_ctl = beta_from_ctl;
    a.feed_pcc = feed_pcc;
    // observables of the incoming state ride on this sweep's k_bonds unless they are switched off (and the
    // PCC controller does not need them) or already on their way
    const bool with_obs = feed_pcc || (s->obs_mode == XY_OBS_ALL && s->obs_valid_T != s->T);
    a.obs_fill = (with_obs && s->obs_valid_T != s->T) ? 1 : 0;
    if (s->timing) {
        if (s->ev_used >= (kTimedKernels + 1) * kTimedSweepsPerFlush)
            if (int rc = timing_flush(s)) return rc;
        if (int rc = timing_mark(s)) return rc;
    }
    if (with_obs) CUDA_TRY(s->ker.bonds(a, 0, s->fourier(), s->grid_bonds, s->stream));
    else CUDA_TRY(s->ker.bonds(a, 2, false, s->grid_bonds_noobs, s->stream));
    if (s->timing) if (int rc = timing_mark(s)) return rc;
    s->ker.label(a, s->stream);
    if (s->timing) if (int rc = timing_mark(s)) return rc;
    s->ker.merge(a, s->stream);
    if (s->timing) if (int rc = timing_mark(s)) return rc;
    s->ker.flip(a, s->grid_fl, s->stream);
    if (s->timing) if (int rc = timing_mark(s)) return rc;
    CUDA_TRY(cudaGetLastError());
    s->launches += 4;
    if (a.obs_fill) s->obs_valid_T = s->T;
    s->T += 1;
    if (s->T - s->oldest_T >= kRingCap) s->oldest_T = s->T - kRingCap + 1;
    s->have_sweep = true;
    s->labels_flat = false;
    return XY_OK;
}

}  // namespace

extern "C" {

const char *xy_last_error(void) { return g_err; }

int xy_workspace_bytes(uint32_t L, uint32_t flags, size_t *nbytes)
{
    if (!nbytes) return fail(XY_ERR_ARG, "nbytes is NULL");
    if (int rc = check_L(L)) return rc;
    if (flags & ~(uint32_t)(XY_FLAG_LABELS64 | XY_FLAG_FOURIER)) return fail(XY_ERR_ARG, "unknown flags 0x%x", flags);
    *nbytes = make_layout(L, flags).total;
    return XY_OK;
}

static int check_slab(uint32_t L, uint32_t rows, uint32_t y_off, uint32_t flags)
{
    if (rows < 32 || rows % 32 != 0 || y_off % 32 != 0 || (uint64_t)y_off + rows > L)
        return fail(XY_ERR_ARG, "slab rows [%u, %u + %u) must be multiples of 32 inside 0..%u", y_off, y_off, rows, L);
    if ((uint64_t)rows * L >= 0x80000000ull) return fail(XY_ERR_ARG, "a slab holds fewer than 2^31 sites (u32 labels with one flag bit)");
    if (flags & XY_FLAG_LABELS64) return fail(XY_ERR_ARG, "slabs use 32-bit labels");
    if (flags & XY_FLAG_FOURIER) return fail(XY_ERR_ARG, "slabs do not reduce the structure-factor sums");
    return XY_OK;
}

static int create_common(xy_state **out, uint32_t L, uint32_t rows, uint32_t y_off, bool slab, uint64_t seed, int init,
                         uint32_t flags, void *dev_workspace, size_t nbytes)
{
    if (!out) return fail(XY_ERR_ARG, "out is NULL");
    *out = nullptr;
    if (int rc = check_L(L)) return rc;
    if (init != XY_INIT_COLD && init != XY_INIT_HOT) return fail(XY_ERR_ARG, "init=%d unknown", init);
    if (flags & ~(uint32_t)(XY_FLAG_LABELS64 | XY_FLAG_FOURIER)) return fail(XY_ERR_ARG, "unknown flags 0x%x", flags);
    if (slab) if (int rc = check_slab(L, rows, y_off, flags)) return rc;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0)
        return fail(XY_ERR_CUDA, "no CUDA device: this library has no CPU fallback");
    xy_state *s = new (std::nothrow) xy_state;
    if (!s) return fail(XY_ERR_NOMEM, "host allocation failed");
    s->L = L; s->rows = rows; s->y_off = y_off; s->slab = slab;
    s->N = (uint64_t)rows * L; s->seed = seed; s->flags = flags;
    s->lay = make_layout(L, flags, rows, slab);
    s->ker = pick_kernels(L, s->l64());
    cudaGetDevice(&s->device);
    if (dev_workspace) {
        if (nbytes < s->lay.total || ((uintptr_t)dev_workspace & 255u)) {
            delete s;
            return fail(XY_ERR_ARG, "workspace too small (%zu < %zu) or not 256-byte aligned", nbytes, make_layout(L, flags, rows, slab).total);
        }
        s->ws = static_cast<char *>(dev_workspace);
    } else {
        void *p = nullptr;
        cudaError_t e = cudaMalloc(&p, s->lay.total);
        if (e != cudaSuccess) {
            const size_t want = s->lay.total;
            delete s;
            cudaGetLastError();
            return fail(XY_ERR_NOMEM, "cudaMalloc(%zu) failed: %s", want, cudaGetErrorString(e));
        }
        s->ws = static_cast<char *>(p);
        s->owns_ws = true;
    }
    if (slab) set_stitch(s, s->ws + s->lay.stitch, default_ranks(L, rows));   // no allocation in the sweep loop
    int bo = 0, bn = 0, fl = 0, sms = 0;
    cudaError_t e = (cudaError_t)s->ker.prepare(s->fourier(), &bo, &bn, &fl);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, s->device);
    if (e != cudaSuccess || bo < 1 || bn < 1 || fl < 1) {
        if (s->owns_ws) cudaFree(s->ws);
        delete s;
        return fail(XY_ERR_CUDA, "kernel occupancy query failed: %s (was the library built for this GPU's sm_100a?)",
                    cudaGetErrorString(e));
    }
    const uint32_t ntiles = (L / s->ker.tw) * (rows / s->ker.th);
    const uint32_t nstrips = (L / s->ker.tw) * (rows / s->ker.rs);
    // the variants of k_bonds with observables share ONE grid so that their fixed-order sums agree bitwise
    long need = (nstrips + BondsShape<true>::warps - 1) / BondsShape<true>::warps;
    long g = (long)sms * bo;
    if (g > need) g = need;
    if (g > (long)kMaxGrid) g = kMaxGrid;
    s->grid_bonds = (int)g;
    need = (nstrips + BondsShape<false>::warps - 1) / BondsShape<false>::warps;
    g = (long)sms * bn;
    if (g > need) g = need;
    if (g > (long)kMaxGrid) g = kMaxGrid;
    s->grid_bonds_noobs = (int)g;
    g = (long)sms * fl;
    if (g > (long)ntiles) g = ntiles;
    s->grid_fl = (int)g;

    // table (cos, sin)(k / 1024), k = 0..kTabN: the angles are exact doubles, the values correctly rounded
    // from the host's long-double libm
    {
        std::vector<double2> h(kTabN + 1);
        for (int k = 0; k <= kTabN; ++k) {
            const long double ang = (long double)k / 1024.0L;
            h[k].x = (double)cosl(ang);
            h[k].y = (double)sinl(ang);
        }
        e = cudaMemcpy(s->tab(), h.data(), h.size() * sizeof(double2), cudaMemcpyHostToDevice);
        if (e != cudaSuccess) {
            if (s->owns_ws) cudaFree(s->ws);
            delete s;
            return fail(XY_ERR_CUDA, "table upload failed: %s", cudaGetErrorString(e));
        }
    }

    if (init == XY_INIT_COLD) {
        e = cudaMemsetAsync(s->theta(), 0, (s->N + (slab ? L : 0)) * 4, nullptr);
    } else {
        k_init_hot<<<148 * 8, 256>>>(s->theta(), s->N, (uint64_t)y_off * L, (uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32));
        // halo row of a slab: the initial values of the row below it in the whole lattice (the draws are keyed by the
        // global site index), so the slab is complete before the caller's first exchange
        if (slab) k_init_hot<<<(L + 255) / 256, 256>>>(s->theta() + s->N, L, (uint64_t)((y_off + rows) % L) * L,
                                                       (uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32));
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) {
        k_ctl_init<<<1, 32>>>(s->ctl(), s->ring(), kRingCap, 0);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(nullptr);
    if (e != cudaSuccess) {
        if (s->owns_ws) cudaFree(s->ws);
        delete s;
        return fail(XY_ERR_CUDA, "initialisation failed: %s", cudaGetErrorString(e));
    }
    *out = s;
    return XY_OK;
}

int xy_create_ex(xy_state **out, uint32_t L, uint64_t seed, int init, uint32_t flags, void *dev_workspace, size_t nbytes)
{
    return create_common(out, L, L, 0, false, seed, init, flags, dev_workspace, nbytes);
}

int xy_create(xy_state **out, uint32_t L, uint64_t seed, int init)
{
    return xy_create_ex(out, L, seed, init, 0, nullptr, 0);
}

int xy_destroy(xy_state *s)
{
    if (!s) return XY_OK;
    DeviceGuard g(s->device);
    cudaStreamSynchronize(s->stream);
    for (cudaEvent_t e : s->ev) cudaEventDestroy(e);
    if (s->stage) cudaFree(s->stage);
    if (s->stitch_owned) cudaFree(s->stitch.key);
    if (s->owns_ws) cudaFree(s->ws);
    delete s;
    return XY_OK;
}

int xy_debug_kernel_timing(xy_state *s, int on)
{
    if (!s) return fail(XY_ERR_ARG, "state is NULL");
    DeviceGuard g(s->device);
    if (int rc = timing_flush(s)) return rc;
    s->timing = on != 0;
    if (on) for (int j = 0; j < kTimedKernels; ++j) { s->t_ms[j] = 0; s->t_n[j] = 0; }
    return XY_OK;
}

int xy_get_kernel_times(xy_state *s, double ms[4], uint64_t launches[4])
{
    if (!s || !ms || !launches) return fail(XY_ERR_ARG, "NULL argument");
    DeviceGuard g(s->device);
    if (int rc = timing_flush(s)) return rc;
    for (int j = 0; j < kTimedKernels; ++j) { ms[j] = s->t_ms[j]; launches[j] = s->t_n[j]; s->t_ms[j] = 0; s->t_n[j] = 0; }
    return XY_OK;
}

int xy_get_launch_count(xy_state *s, uint64_t *count)
{
    if (!s || !count) return fail(XY_ERR_ARG, "NULL argument");
    *count = s->launches;
    return XY_OK;
}

int xy_sw_sweeps(xy_state *s, double beta, uint64_t n, void *cuda_stream)
{
    if (!s) return fail(XY_ERR_ARG, "state is NULL");
    if (!(beta >= 0.0) || !std::isfinite(beta)) return fail(XY_ERR_ARG, "beta must be finite and >= 0");
    if (s->T + n > 0xffffffffull) return fail(XY_ERR_STATE, "sweep counter would reach 2^32");
    if (s->slab) return fail(XY_ERR_STATE, "a slab sweeps with xy_slab_label / xy_slab_flip (an exchange lies between them)");
    DeviceGuard g(s->device);
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    if (st != s->stream) {
        // keep stream order across a change of stream
        CUDA_TRY(cudaStreamSynchronize(s->stream));
        s->stream = st;
    }
    for (uint64_t k = 0; k < n; ++k)
        if (int rc = enqueue_sweep(s, beta, 0, 0)) return rc;
    return XY_OK;
}

int xy_measure(xy_state *s, xy_obs *out)
{
    if (!s || !out) return fail(XY_ERR_ARG, "NULL argument");
    DeviceGuard g(s->device);
    if (int rc = ensure_obs(s, 0)) return rc;
    CUDA_TRY(cudaMemcpyAsync(out, s->ring() + (s->T % kRingCap), sizeof(xy_obs), cudaMemcpyDeviceToHost, s->stream));
    CUDA_TRY(cudaStreamSynchronize(s->stream));
    return slab_stitch_check(s);
}

static int pcc_loop(xy_state *s, double beta0, double dbeta0, const xy_pcc_schedule *sc, xy_pcc_out *out, bool fresh)
{
    if (!s || !sc || !out) return fail(XY_ERR_ARG, "NULL argument");
    if (fresh && (!(beta0 >= 0.0) || !std::isfinite(beta0) || !(dbeta0 >= 0.0) || !std::isfinite(dbeta0)))
        return fail(XY_ERR_ARG, "beta0 and dbeta0 must be finite and >= 0");
    if (sc->window < 1 || (sc->dirs != 1 && sc->dirs != 2)) return fail(XY_ERR_ARG, "window must be >= 1 and dirs 1 or 2");
    if (sc->discard > sc->n_sweeps) return fail(XY_ERR_ARG, "discard > n_sweeps");
    if (s->T + sc->n_sweeps > 0xffffffffull) return fail(XY_ERR_STATE, "sweep counter would reach 2^32");
    if (s->slab) return fail(XY_ERR_STATE, "the PCC controller needs the sums of the whole lattice: not available on a slab");
    DeviceGuard g(s->device);
    // measured sweeps the controller has been fed before this call (0 for a fresh run)
    uint64_t k0 = 0;
    if (!fresh) {
        DevCtl h0;
        CUDA_TRY(cudaMemcpyAsync(&h0, s->ctl(), sizeof h0, cudaMemcpyDeviceToHost, s->stream));
        CUDA_TRY(cudaStreamSynchronize(s->stream));
        k0 = h0.k;
    }
    const uint64_t measured = sc->n_sweeps - sc->discard;
    const uint64_t max_dec = (k0 + measured) / sc->window - k0 / sc->window;
    double *d_trace = nullptr;
    if (max_dec > 0) CUDA_TRY(cudaMalloc(&d_trace, max_dec * 2 * sizeof(double)));
    PccSetup ps;
    ps.beta0 = beta0; ps.dbeta0 = dbeta0;
    ps.halve_every = sc->halve_every; ps.dbeta_min = sc->dbeta_min; ps.target = sc->target;
    ps.window = sc->window; ps.dirs = sc->dirs;
    ps.trace_beta = d_trace; ps.trace_bY = d_trace ? d_trace + max_dec : nullptr; ps.trace_cap = max_dec;
    k_pcc_setup<<<1, 32, 0, s->stream>>>(s->ctl(), ps, fresh ? 1 : 0);
    int rc = XY_OK;
    bool feed_next = false;        // the next k_bonds feeds the record of the incoming state
    for (uint64_t n = 0; n < sc->n_sweeps && rc == XY_OK; ++n) {
        rc = enqueue_sweep(s, beta0, 1, feed_next ? 1 : 0);
        feed_next = false;
        if (rc != XY_OK || n < sc->discard) continue;
        const uint64_t k = k0 + n - sc->discard + 1;
        const bool decision = (k % sc->window) == 0;
        if (decision || n + 1 == sc->n_sweeps) rc = ensure_obs(s, 1);   // beta must move before the next sweep reads it
        else feed_next = true;
    }
    DevCtl h;
    if (rc == XY_OK) {
        cudaError_t e = cudaMemcpyAsync(&h, s->ctl(), sizeof h, cudaMemcpyDeviceToHost, s->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
        const uint64_t ndec = e == cudaSuccess ? h.n_dec - h.trace_base : 0;
        if (e == cudaSuccess && d_trace && out->trace_beta && out->trace_bY && out->trace_cap) {
            const uint64_t ncopy = ndec < out->trace_cap ? ndec : out->trace_cap;
            e = cudaMemcpy(out->trace_beta, d_trace, ncopy * sizeof(double), cudaMemcpyDeviceToHost);
            if (e == cudaSuccess) e = cudaMemcpy(out->trace_bY, d_trace + max_dec, ncopy * sizeof(double), cudaMemcpyDeviceToHost);
        }
        // the trace arrays of this call are about to be freed: the controller must not keep pointers to them
        if (e == cudaSuccess) e = cudaMemsetAsync(&s->ctl()->trace_beta, 0, 2 * sizeof(double *), s->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
        if (e != cudaSuccess) rc = fail(XY_ERR_CUDA, "PCC run failed: %s", cudaGetErrorString(e));
    } else {
        cudaStreamSynchronize(s->stream);
    }
    if (d_trace) cudaFree(d_trace);
    if (rc != XY_OK) return rc;
    out->beta_final = h.beta;
    out->dbeta_final = h.dbeta;
    out->n_decisions = h.n_dec - h.trace_base;
    out->trace_len = h.n_dec - h.trace_base;
    if (h.stage_cnt > 0) out->beta_mean = h.stage_sum / (double)h.stage_cnt;
    else if (h.last_cnt > 0) out->beta_mean = h.last_sum / (double)h.last_cnt;
    else out->beta_mean = h.beta;
    return XY_OK;
}

int xy_pcc_run(xy_state *s, double beta0, double dbeta0, const xy_pcc_schedule *sc, xy_pcc_out *out)
{
    return pcc_loop(s, beta0, dbeta0, sc, out, true);
}

int xy_pcc_continue(xy_state *s, const xy_pcc_schedule *sc, xy_pcc_out *out)
{
    return pcc_loop(s, 0.0, 0.0, sc, out, false);
}

int xy_pcc_get_state(xy_state *s, xy_pcc_state *out)
{
    if (!s || !out) return fail(XY_ERR_ARG, "NULL argument");
    DeviceGuard g(s->device);
    DevCtl h;
    CUDA_TRY(cudaMemcpyAsync(&h, s->ctl(), sizeof h, cudaMemcpyDeviceToHost, s->stream));
    CUDA_TRY(cudaStreamSynchronize(s->stream));
    out->beta = h.beta; out->dbeta = h.dbeta; out->acc_e = h.acc_e; out->acc_s2 = h.acc_s2;
    out->k = h.k; out->n_decisions = h.n_dec;
    out->stage_sum = h.stage_sum; out->last_sum = h.last_sum; out->stage_cnt = h.stage_cnt; out->last_cnt = h.last_cnt;
    out->sum_m2 = h.sum_m2; out->sum_chik = h.sum_chik; out->n_acc = h.n_acc;
    return XY_OK;
}

int xy_pcc_set_state(xy_state *s, const xy_pcc_state *in)
{
    if (!s || !in) return fail(XY_ERR_ARG, "NULL argument");
    if (!(in->beta >= 0.0) || !std::isfinite(in->beta) || !(in->dbeta >= 0.0) || !std::isfinite(in->dbeta))
        return fail(XY_ERR_ARG, "beta and dbeta must be finite and >= 0");
    DeviceGuard g(s->device);
    DevCtl h;
    CUDA_TRY(cudaMemcpyAsync(&h, s->ctl(), sizeof h, cudaMemcpyDeviceToHost, s->stream));
    CUDA_TRY(cudaStreamSynchronize(s->stream));
    h.beta = in->beta; h.dbeta = in->dbeta; h.acc_e = in->acc_e; h.acc_s2 = in->acc_s2;
    h.k = in->k; h.n_dec = in->n_decisions;
    h.stage_sum = in->stage_sum; h.last_sum = in->last_sum; h.stage_cnt = in->stage_cnt; h.last_cnt = in->last_cnt;
    h.sum_m2 = in->sum_m2; h.sum_chik = in->sum_chik; h.n_acc = in->n_acc;
    h.trace_beta = nullptr; h.trace_bY = nullptr; h.trace_cap = 0;
    CUDA_TRY(cudaMemcpyAsync(s->ctl(), &h, sizeof h, cudaMemcpyHostToDevice, s->stream));
    CUDA_TRY(cudaStreamSynchronize(s->stream));
    return XY_OK;
}

static int check_range(const xy_state *s, uint64_t first, size_t n)
{
    if (n == 0 || first >= s->N || n > s->N - first)
        return fail(XY_ERR_ARG, "sites %llu..%llu not in 0..%llu", (unsigned long long)first,
                    (unsigned long long)(first + n) - 1, (unsigned long long)s->N - 1);
    return XY_OK;
}

int xy_get_angles_range(xy_state *s, float *host, uint64_t first, size_t n)
{
    if (!s || !host) return fail(XY_ERR_ARG, "NULL argument");
    if (int rc = check_range(s, first, n)) return rc;
    DeviceGuard g(s->device);
    CUDA_TRY(cudaMemcpyAsync(host, s->theta() + first, n * sizeof(float), cudaMemcpyDeviceToHost, s->stream));
    CUDA_TRY(cudaStreamSynchronize(s->stream));
    return XY_OK;
}

int xy_get_angles(xy_state *s, float *host, size_t n) { return xy_get_angles_range(s, host, 0, n); }

int xy_set_angles(xy_state *s, const float *host, size_t n)
{
    if (!s || !host) return fail(XY_ERR_ARG, "NULL argument");
    if (n != s->N) return fail(XY_ERR_ARG, "n=%zu but L*L=%llu", n, (unsigned long long)s->N);
    if (s->slab_labelled) return fail(XY_ERR_STATE, "xy_slab_flip is pending: its labels live where the angles would be staged");
    DeviceGuard g(s->device);
    // staged in the label array (>= 4 N bytes; the labels of the previous sweep are given up), checked
    // there, and copied to theta only if every value is in range: a rejected call leaves theta untouched
    float *stage = static_cast<float *>(s->labels());
    CUDA_TRY(cudaMemcpyAsync(stage, host, n * sizeof(float), cudaMemcpyHostToDevice, s->stream));
    k_check_angles<<<148 * 8, 256, 0, s->stream>>>(stage, s->N, &s->ctl()->pad);
    unsigned int bad = 0;
    CUDA_TRY(cudaMemcpyAsync(&bad, &s->ctl()->pad, sizeof bad, cudaMemcpyDeviceToHost, s->stream));
    CUDA_TRY(cudaStreamSynchronize(s->stream));
    s->have_sweep = false;
    if (bad) {
        CUDA_TRY(cudaMemsetAsync(&s->ctl()->pad, 0, sizeof bad, s->stream));
        return fail(XY_ERR_ARG, "angles outside [0, 6.2831855] (or NaN): rejected, the configuration is unchanged");
    }
    CUDA_TRY(cudaMemcpyAsync(s->theta(), stage, n * sizeof(float), cudaMemcpyDeviceToDevice, s->stream));
    k_ring_reset<<<1, 32, 0, s->stream>>>(s->ring(), kRingCap, s->T);
    CUDA_TRY(cudaStreamSynchronize(s->stream));
    s->obs_valid_T = UINT64_MAX;
    s->oldest_T = s->T;
    return XY_OK;
}

int xy_set_obs_mode(xy_state *s, int mode)
{
    if (!s) return fail(XY_ERR_ARG, "state is NULL");
    if (mode != XY_OBS_NONE && mode != XY_OBS_ALL) return fail(XY_ERR_ARG, "obs mode %d unknown", mode);
    s->obs_mode = mode;
    return XY_OK;
}

int xy_get_sweep(xy_state *s, uint64_t *t)
{
    if (!s || !t) return fail(XY_ERR_ARG, "NULL argument");
    *t = s->T;
    return XY_OK;
}

int xy_set_sweep(xy_state *s, uint64_t t)
{
    if (!s) return fail(XY_ERR_ARG, "state is NULL");
    if (t > 0xffffffffull) return fail(XY_ERR_STATE, "sweep counter must stay below 2^32");
    DeviceGuard g(s->device);
    s->T = t;
    k_ring_reset<<<1, 32, 0, s->stream>>>(s->ring(), kRingCap, s->T);
    CUDA_TRY(cudaStreamSynchronize(s->stream));
    s->obs_valid_T = UINT64_MAX;
    s->oldest_T = t;
    s->have_sweep = false;
    return XY_OK;
}

int xy_debug_fix_phi(xy_state *s, int on, double phi)
{
    if (!s) return fail(XY_ERR_ARG, "state is NULL");
    if (on && !std::isfinite(phi)) return fail(XY_ERR_ARG, "phi must be finite");
    s->fix_phi = on != 0;
    s->phi_fixed = phi;
    return XY_OK;
}

int xy_series_capacity(xy_state *s, uint64_t *cap)
{
    if (!s || !cap) return fail(XY_ERR_ARG, "NULL argument");
    *cap = kRingCap;
    return XY_OK;
}

int xy_get_series(xy_state *s, xy_obs *host, uint64_t first, uint64_t count)
{
    if (!s || (!host && count)) return fail(XY_ERR_ARG, "NULL argument");
    if (count == 0) return XY_OK;
    if (first < s->oldest_T || first + count - 1 > s->T)
        return fail(XY_ERR_ARG, "records %llu..%llu not in the ring (holds %llu..%llu)", (unsigned long long)first,
                    (unsigned long long)(first + count - 1), (unsigned long long)s->oldest_T, (unsigned long long)s->T);
    DeviceGuard g(s->device);
    if (first + count - 1 == s->T)
        if (int rc = ensure_obs(s, 0)) return rc;
    uint64_t done = 0;
    while (done < count) {
        const uint64_t slot = (first + done) % kRingCap;
        uint64_t run = kRingCap - slot;
        if (run > count - done) run = count - done;
        CUDA_TRY(cudaMemcpyAsync(host + done, s->ring() + slot, run * sizeof(xy_obs), cudaMemcpyDeviceToHost, s->stream));
        done += run;
    }
    CUDA_TRY(cudaStreamSynchronize(s->stream));
    return XY_OK;
}

int xy_measure_fourier(xy_state *s, xy_fourier *out)
{
    if (!s || !out) return fail(XY_ERR_ARG, "NULL argument");
    if (!s->fourier()) return fail(XY_ERR_STATE, "state was created without XY_FLAG_FOURIER");
    DeviceGuard g(s->device);
    if (int rc = ensure_obs(s, 0)) return rc;
    CUDA_TRY(cudaMemcpyAsync(out, s->fring() + (s->T % kRingCap), sizeof(xy_fourier), cudaMemcpyDeviceToHost, s->stream));
    CUDA_TRY(cudaStreamSynchronize(s->stream));
    return XY_OK;
}

int xy_get_fourier_series(xy_state *s, xy_fourier *host, uint64_t first, uint64_t count)
{
    if (!s || (!host && count)) return fail(XY_ERR_ARG, "NULL argument");
    if (!s->fourier()) return fail(XY_ERR_STATE, "state was created without XY_FLAG_FOURIER");
    if (count == 0) return XY_OK;
    if (first < s->oldest_T || first + count - 1 > s->T)
        return fail(XY_ERR_ARG, "records %llu..%llu not in the ring (holds %llu..%llu)", (unsigned long long)first,
                    (unsigned long long)(first + count - 1), (unsigned long long)s->oldest_T, (unsigned long long)s->T);
    DeviceGuard g(s->device);
    if (first + count - 1 == s->T)
        if (int rc = ensure_obs(s, 0)) return rc;
    uint64_t done = 0;
    while (done < count) {
        const uint64_t slot = (first + done) % kRingCap;
        uint64_t run = kRingCap - slot;
        if (run > count - done) run = count - done;
        CUDA_TRY(cudaMemcpyAsync(host + done, s->fring() + slot, run * sizeof(xy_fourier), cudaMemcpyDeviceToHost, s->stream));
        done += run;
    }
    CUDA_TRY(cudaStreamSynchronize(s->stream));
    return XY_OK;
}

int xy_xi2nd(double chi0, double chik, uint32_t L, double *out)
{
    if (!out) return fail(XY_ERR_ARG, "out is NULL");
    *out = std::numeric_limits<double>::quiet_NaN();
    if (L < 2 || !std::isfinite(chi0) || !std::isfinite(chik) || !(chik > 0.0) || !(chi0 >= chik))
        return fail(XY_ERR_ARG, "xi_2nd needs L >= 2 and finite chi(0) >= chi(2 pi / L) > 0");
    *out = std::sqrt(chi0 / chik - 1.0) / (2.0 * std::sin(kPi / (double)L));
    return XY_OK;
}

int xy_debug_check_counts(uint64_t counts[8], int *checked_build)
{
    if (!counts || !checked_build) return fail(XY_ERR_ARG, "NULL argument");
    for (int k = 0; k < 8; ++k) counts[k] = 0;
#ifdef XY_CHECKED
    *checked_build = 1;
    unsigned long long h[8];
    CUDA_TRY(cudaDeviceSynchronize());
    CUDA_TRY(cudaMemcpyFromSymbol(h, g_xy_check_fail, sizeof h));
    for (int k = 0; k < 8; ++k) counts[k] = h[k];
#else
    *checked_build = 0;
#endif
    return XY_OK;
}

int xy_get_fallback_count(xy_state *s, uint64_t *count)
{
    if (!s || !count) return fail(XY_ERR_ARG, "NULL argument");
    DeviceGuard g(s->device);
    unsigned long long v = 0;
    CUDA_TRY(cudaMemcpyAsync(&v, &s->ctl()->fallback_count, sizeof v, cudaMemcpyDeviceToHost, s->stream));
    CUDA_TRY(cudaStreamSynchronize(s->stream));
    *count = v;
    return XY_OK;
}

// label[i] <- root(i) in place, once per sweep (S5 as an array; the sweep itself never needs it)
static int ensure_flat(xy_state *s)
{
    if (s->labels_flat) return XY_OK;
    if (s->l64()) k_flatten<uint64_t><<<148 * 8, 256, 0, s->stream>>>(static_cast<uint64_t *>(s->labels()), s->N);
    else k_flatten<uint32_t><<<148 * 8, 256, 0, s->stream>>>(static_cast<uint32_t *>(s->labels()), s->N);
    CUDA_TRY(cudaGetLastError());
    s->launches += 1;
    s->labels_flat = true;
    return XY_OK;
}

int xy_get_labels_range(xy_state *s, int64_t *host, uint64_t first, size_t n)
{
    if (!s || !host) return fail(XY_ERR_ARG, "NULL argument");
    if (int rc = check_range(s, first, n)) return rc;
    if (!s->have_sweep) return fail(XY_ERR_STATE, "no sweep has produced labels yet");
    DeviceGuard g(s->device);
    if (int rc = ensure_stage(s)) return rc;
    if (s->slab) {
        // canonical labels of the whole lattice; valid after xy_slab_flip (the stitch overrides are in place)
        if (s->slab_labelled) return fail(XY_ERR_STATE, "labels of a slab are complete after xy_slab_flip");
        if (int rc = slab_stitch_check(s)) return rc;
        const uint64_t chunk = kStageBytes / sizeof(int64_t);
        for (uint64_t done = 0; done < n; done += chunk) {
            const uint64_t m = n - done < chunk ? n - done : chunk;
            k_slab_labels_to_i64<<<148 * 4, 256, 0, s->stream>>>(static_cast<const uint32_t *>(s->labels()), s->xroot(),
                                                                 (uint64_t)s->y_off * s->L, static_cast<int64_t *>(s->stage), first + done, m);
            CUDA_TRY(cudaMemcpyAsync(host + done, s->stage, m * sizeof(int64_t), cudaMemcpyDeviceToHost, s->stream));
            CUDA_TRY(cudaStreamSynchronize(s->stream));
        }
        return XY_OK;
    }
    if (int rc = ensure_flat(s)) return rc;
    const uint64_t chunk = kStageBytes / sizeof(int64_t);
    for (uint64_t done = 0; done < n; done += chunk) {
        const uint64_t m = n - done < chunk ? n - done : chunk;
        if (s->l64()) k_labels_to_i64<uint64_t><<<148 * 4, 256, 0, s->stream>>>(static_cast<const uint64_t *>(s->labels()), static_cast<int64_t *>(s->stage), first + done, m);
        else k_labels_to_i64<uint32_t><<<148 * 4, 256, 0, s->stream>>>(static_cast<const uint32_t *>(s->labels()), static_cast<int64_t *>(s->stage), first + done, m);
        CUDA_TRY(cudaMemcpyAsync(host + done, s->stage, m * sizeof(int64_t), cudaMemcpyDeviceToHost, s->stream));
        CUDA_TRY(cudaStreamSynchronize(s->stream));
    }
    return XY_OK;
}

int xy_get_labels(xy_state *s, int64_t *host, size_t n) { return xy_get_labels_range(s, host, 0, n); }

int xy_debug_check_labels(xy_state *s, uint64_t counts[5])
{
    if (!s || !counts) return fail(XY_ERR_ARG, "NULL argument");
    if (!s->have_sweep) return fail(XY_ERR_STATE, "no sweep has produced labels yet");
    if (s->slab) return fail(XY_ERR_STATE, "not available on a slab");
    DeviceGuard g(s->device);
    if (int rc = ensure_stage(s)) return rc;
    if (int rc = ensure_flat(s)) return rc;
    unsigned long long *d = static_cast<unsigned long long *>(s->stage);
    CUDA_TRY(cudaMemsetAsync(d, 0, 5 * sizeof(unsigned long long), s->stream));
    if (s->l64()) k_check_labels<uint64_t><<<148 * 8, 256, 0, s->stream>>>(static_cast<const uint64_t *>(s->labels()), s->bonds(), s->L, d);
    else k_check_labels<uint32_t><<<148 * 8, 256, 0, s->stream>>>(static_cast<const uint32_t *>(s->labels()), s->bonds(), s->L, d);
    CUDA_TRY(cudaGetLastError());
    s->launches += 1;
    unsigned long long h[5];
    CUDA_TRY(cudaMemcpyAsync(h, d, sizeof h, cudaMemcpyDeviceToHost, s->stream));
    CUDA_TRY(cudaStreamSynchronize(s->stream));
    for (int k = 0; k < 5; ++k) counts[k] = h[k];
    return XY_OK;
}

int xy_get_bonds_range(xy_state *s, uint8_t *host, uint64_t first, size_t n)
{
    if (!s || !host) return fail(XY_ERR_ARG, "NULL argument");
    if (int rc = check_range(s, first, n)) return rc;
    if (!s->have_sweep) return fail(XY_ERR_STATE, "no sweep has produced bonds yet");
    DeviceGuard g(s->device);
    if (int rc = ensure_stage(s)) return rc;
    const uint64_t chunk = kStageBytes;
    for (uint64_t done = 0; done < n; done += chunk) {
        const uint64_t m = n - done < chunk ? n - done : chunk;
        k_bonds_unpack<<<148 * 4, 256, 0, s->stream>>>(s->bonds(), static_cast<uint8_t *>(s->stage), first + done, m);
        CUDA_TRY(cudaMemcpyAsync(host + done, s->stage, m, cudaMemcpyDeviceToHost, s->stream));
        CUDA_TRY(cudaStreamSynchronize(s->stream));
    }
    return XY_OK;
}

int xy_get_bonds(xy_state *s, uint8_t *host, size_t n) { return xy_get_bonds_range(s, host, 0, n); }

int xy_label_bonds(xy_state *s, const uint8_t *host_bonds, size_t n)
{
    if (!s || !host_bonds) return fail(XY_ERR_ARG, "NULL argument");
    if (n != s->N) return fail(XY_ERR_ARG, "n=%zu but L*L=%llu", n, (unsigned long long)s->N);
    if (s->slab) return fail(XY_ERR_STATE, "not available on a slab");
    DeviceGuard g(s->device);
    if (int rc = ensure_stage(s)) return rc;
    const uint64_t chunk = kStageBytes;            // canonical bytes per pass (multiple of 4)
    for (uint64_t first = 0; first < s->N; first += chunk) {
        const uint64_t m = s->N - first < chunk ? s->N - first : chunk;
        CUDA_TRY(cudaMemcpyAsync(s->stage, host_bonds + first, m, cudaMemcpyHostToDevice, s->stream));
        k_bonds_pack<<<148 * 4, 256, 0, s->stream>>>(static_cast<const uint8_t *>(s->stage), s->bonds(), first / 4, m / 4);
        CUDA_TRY(cudaStreamSynchronize(s->stream));
    }
    SweepArgs a = base_args(s);
    cudaEvent_t ev[3] = {nullptr, nullptr, nullptr};
    if (s->timing) {
        if (int rc = timing_flush(s)) return rc;
        for (auto &e : ev) CUDA_TRY(cudaEventCreate(&e));
        CUDA_TRY(cudaEventRecord(ev[0], s->stream));
    }
    s->ker.label(a, s->stream);
    if (s->timing) CUDA_TRY(cudaEventRecord(ev[1], s->stream));
    s->ker.merge(a, s->stream);
    if (s->timing) CUDA_TRY(cudaEventRecord(ev[2], s->stream));
    s->launches += 2;
    CUDA_TRY(cudaGetLastError());
    CUDA_TRY(cudaStreamSynchronize(s->stream));
    if (s->timing) {                      // labeling-only timings land in the k_label / k_merge accumulators
        for (int j = 0; j < 2; ++j) {
            float ms = 0;
            CUDA_TRY(cudaEventElapsedTime(&ms, ev[j], ev[j + 1]));
            s->t_ms[1 + j] += ms;
            s->t_n[1 + j] += 1;
        }
        for (auto &e : ev) cudaEventDestroy(e);
    }
    s->have_sweep = true;
    s->labels_flat = false;
    return XY_OK;
}

static int debug_philox_common(const uint32_t *ctr, const uint32_t *key, uint32_t *out, size_t n, bool curand_fn)
{
    if (!ctr || !key || !out) return fail(XY_ERR_ARG, "NULL argument");
    if (n == 0) return XY_OK;
    uint32_t *d = nullptr;
    CUDA_TRY(cudaMalloc(&d, n * 10 * sizeof(uint32_t)));
    cudaError_t e = cudaMemcpy(d, ctr, n * 16, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(d + 4 * n, key, n * 8, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        const unsigned blocks = (unsigned)((n + 255) / 256);
        if (curand_fn) k_debug_curand_philox<<<blocks, 256>>>(d, d + 4 * n, d + 6 * n, n);
        else k_debug_philox<<<blocks, 256>>>(d, d + 4 * n, d + 6 * n, n);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpy(out, d + 6 * n, n * 16, cudaMemcpyDeviceToHost);
    cudaFree(d);
    if (e != cudaSuccess) return fail(XY_ERR_CUDA, "debug philox failed: %s", cudaGetErrorString(e));
    return XY_OK;
}

// ---------------------------------------------------------------------------------------------
// Row-slab sharding: one state per rank holds rows [y_off, y_off + rows).
// ---------------------------------------------------------------------------------------------
int xy_slab_workspace_bytes(uint32_t L, uint32_t rows, uint32_t flags, size_t *nbytes)
{
    if (!nbytes) return fail(XY_ERR_ARG, "nbytes is NULL");
    if (int rc = check_L(L)) return rc;
    if (flags & ~(uint32_t)(XY_FLAG_LABELS64 | XY_FLAG_FOURIER)) return fail(XY_ERR_ARG, "unknown flags 0x%x", flags);
    if (int rc = check_slab(L, rows, 0, flags)) return rc;
    *nbytes = make_layout(L, flags, rows, true).total;
    return XY_OK;
}

int xy_slab_create(xy_state **out, uint32_t L, uint32_t rows, uint32_t y_off, uint64_t seed, int init, uint32_t flags,
                   void *dev_workspace, size_t nbytes)
{
    return create_common(out, L, rows, y_off, true, seed, init, flags, dev_workspace, nbytes);
}

int xy_slab_buffers(xy_state *s, void **dev_first_row, void **dev_halo_row, size_t *row_bytes, void **dev_edges, size_t *edge_bytes)
{
    if (!s || !dev_first_row || !dev_halo_row || !row_bytes || !dev_edges || !edge_bytes) return fail(XY_ERR_ARG, "NULL argument");
    if (!s->slab) return fail(XY_ERR_STATE, "not a slab");
    *dev_first_row = s->theta();
    *dev_halo_row = s->theta() + s->N;
    *row_bytes = (size_t)s->L * sizeof(float);
    *dev_edges = s->edges();
    *edge_bytes = slab_edge_bytes(s->L);
    return XY_OK;
}

static int slab_label_common(xy_state *s, double beta, int beta_from_ctl, void *cuda_stream)
{
    if (!s) return fail(XY_ERR_ARG, "state is NULL");
    if (!s->slab) return fail(XY_ERR_STATE, "not a slab");
    if (s->slab_labelled) return fail(XY_ERR_STATE, "xy_slab_flip of the previous xy_slab_label is pending");
    if (!beta_from_ctl && (!(beta >= 0.0) || !std::isfinite(beta))) return fail(XY_ERR_ARG, "beta must be finite and >= 0");
    if (s->T >= 0xffffffffull) return fail(XY_ERR_STATE, "sweep counter would reach 2^32");
    DeviceGuard g(s->device);
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    if (st != s->stream) {
        CUDA_TRY(cudaStreamSynchronize(s->stream));
        s->stream = st;
    }
    SweepArgs a = base_args(s);
    set_direction(s, s->T, a);
    a.beta = beta;
    a.beta_from_ctl = beta_from_ctl;
    const bool with_obs = s->obs_mode == XY_OBS_ALL && s->obs_valid_T != s->T;
    a.obs_fill = with_obs ? 1 : 0;
    if (with_obs) CUDA_TRY(s->ker.bonds(a, 0, s->fourier(), s->grid_bonds, s->stream));
    else CUDA_TRY(s->ker.bonds(a, 2, false, s->grid_bonds_noobs, s->stream));
    s->ker.label(a, s->stream);
    s->ker.merge(a, s->stream);
    k_slab_edges<<<(s->L + 255) / 256, 256, 0, s->stream>>>(static_cast<const uint32_t *>(s->labels()), s->bonds(), s->L,
                                                           s->rows, s->y_off, s->edges());
    CUDA_TRY(cudaGetLastError());
    s->launches += 4;
    if (a.obs_fill) s->obs_valid_T = s->T;
    s->pending = a;
    s->slab_labelled = true;
    return XY_OK;
}

int xy_slab_label(xy_state *s, double beta, void *cuda_stream) { return slab_label_common(s, beta, 0, cuda_stream); }

/* parity hook (the slab counterpart of xy_label_bonds): label an injected bond set of the slab's sites */
int xy_slab_label_bonds(xy_state *s, const uint8_t *host_bonds, size_t n)
{
    if (!s || !host_bonds) return fail(XY_ERR_ARG, "NULL argument");
    if (!s->slab) return fail(XY_ERR_STATE, "not a slab");
    if (n != s->N) return fail(XY_ERR_ARG, "n=%zu but the slab holds %llu sites", n, (unsigned long long)s->N);
    if (s->slab_labelled) return fail(XY_ERR_STATE, "xy_slab_flip of the previous label phase is pending");
    DeviceGuard g(s->device);
    if (int rc = ensure_stage(s)) return rc;
    for (uint64_t first = 0; first < s->N; first += kStageBytes) {
        const uint64_t m = s->N - first < kStageBytes ? s->N - first : kStageBytes;
        CUDA_TRY(cudaMemcpyAsync(s->stage, host_bonds + first, m, cudaMemcpyHostToDevice, s->stream));
        k_bonds_pack<<<148 * 4, 256, 0, s->stream>>>(static_cast<const uint8_t *>(s->stage), s->bonds(), first / 4, m / 4);
        CUDA_TRY(cudaStreamSynchronize(s->stream));
    }
    SweepArgs a = base_args(s);
    set_direction(s, s->T, a);
    a.beta = 0.0;
    s->ker.label(a, s->stream);
    s->ker.merge(a, s->stream);
    k_slab_edges<<<(s->L + 255) / 256, 256, 0, s->stream>>>(static_cast<const uint32_t *>(s->labels()), s->bonds(), s->L,
                                                           s->rows, s->y_off, s->edges());
    CUDA_TRY(cudaGetLastError());
    s->launches += 3;
    s->pending = a;
    s->slab_labelled = true;
    return XY_OK;
}

/* ---- PCC on a sharded lattice: the controller runs replicated on every rank, fed with all-reduced sums ---- */
int xy_slab_pcc_setup(xy_state *s, double beta0, double dbeta0, const xy_pcc_schedule *sc)
{
    if (!s || !sc) return fail(XY_ERR_ARG, "NULL argument");
    if (!s->slab) return fail(XY_ERR_STATE, "not a slab");
    if (!(beta0 >= 0.0) || !std::isfinite(beta0) || !(dbeta0 >= 0.0) || !std::isfinite(dbeta0))
        return fail(XY_ERR_ARG, "beta0 and dbeta0 must be finite and >= 0");
    if (sc->window < 1 || (sc->dirs != 1 && sc->dirs != 2)) return fail(XY_ERR_ARG, "window must be >= 1 and dirs 1 or 2");
    DeviceGuard g(s->device);
    PccSetup ps;
    ps.beta0 = beta0; ps.dbeta0 = dbeta0;
    ps.halve_every = sc->halve_every; ps.dbeta_min = sc->dbeta_min; ps.target = sc->target;
    ps.window = sc->window; ps.dirs = sc->dirs;
    ps.trace_beta = nullptr; ps.trace_bY = nullptr; ps.trace_cap = 0;
    k_pcc_setup<<<1, 32, 0, s->stream>>>(s->ctl(), ps, 1);
    CUDA_TRY(cudaGetLastError());
    return XY_OK;
}

int xy_slab_label_pcc(xy_state *s, void *cuda_stream) { return slab_label_common(s, 0.0, 1, cuda_stream); }

int xy_slab_pcc_buffers(xy_state *s, void **dev_partial8, void **dev_global8)
{
    if (!s || !dev_partial8 || !dev_global8) return fail(XY_ERR_ARG, "NULL argument");
    if (!s->slab) return fail(XY_ERR_STATE, "not a slab");
    *dev_partial8 = s->pccbuf();
    *dev_global8 = s->pccbuf() + 8;
    return XY_OK;
}

int xy_slab_obs_partial(xy_state *s, void *cuda_stream)
{
    if (!s) return fail(XY_ERR_ARG, "state is NULL");
    if (!s->slab) return fail(XY_ERR_STATE, "not a slab");
    if (s->slab_labelled) return fail(XY_ERR_STATE, "xy_slab_flip is pending");
    DeviceGuard g(s->device);
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    if (st != s->stream) { CUDA_TRY(cudaStreamSynchronize(s->stream)); s->stream = st; }
    if (int rc = ensure_obs(s, 0)) return rc;
    k_slab_pack_obs<<<1, 32, 0, s->stream>>>(s->ring() + (s->T % kRingCap), s->pccbuf());
    CUDA_TRY(cudaGetLastError());
    return XY_OK;
}

int xy_slab_pcc_feed(xy_state *s, void *cuda_stream)
{
    if (!s) return fail(XY_ERR_ARG, "state is NULL");
    if (!s->slab) return fail(XY_ERR_STATE, "not a slab");
    DeviceGuard g(s->device);
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    if (st != s->stream) { CUDA_TRY(cudaStreamSynchronize(s->stream)); s->stream = st; }
    k_slab_pcc_feed<<<1, 32, 0, s->stream>>>(s->ctl(), s->pccbuf() + 8, (double)s->L * (double)s->L);
    CUDA_TRY(cudaGetLastError());
    return XY_OK;
}

int xy_slab_flip(xy_state *s, const void *dev_gathered_edges, uint32_t nranks, uint32_t rank, void *cuda_stream)
{
    if (!s || !dev_gathered_edges) return fail(XY_ERR_ARG, "NULL argument");
    if (!s->slab) return fail(XY_ERR_STATE, "not a slab");
    if (!s->slab_labelled) return fail(XY_ERR_STATE, "call xy_slab_label first");
    if (nranks < 1 || rank >= nranks) return fail(XY_ERR_ARG, "rank %u of %u", rank, nranks);
    DeviceGuard g(s->device);
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    if (st != s->stream) {
        CUDA_TRY(cudaStreamSynchronize(s->stream));
        s->stream = st;
    }
    const uint64_t entries = (uint64_t)nranks * 2u * s->L;
    if (entries >= (1ull << 29)) return fail(XY_ERR_ARG, "too many cut sites");
    if (s->stitch_ranks != nranks) {
        // not the number of slabs the workspace table was sized for (create_common): a table of its own
        if (s->stitch_owned) { CUDA_TRY(cudaStreamSynchronize(s->stream)); cudaFree(s->stitch.key); }
        s->stitch = StitchTable{};
        s->stitch_owned = false;
        s->stitch_ranks = 0;
        void *p = nullptr;
        CUDA_TRY(cudaMalloc(&p, stitch_bytes(s->L, nranks)));
        set_stitch(s, p, nranks);
        s->stitch_owned = true;
    }
    const unsigned char *gathered = static_cast<const unsigned char *>(dev_gathered_edges);
    const int grid = 148 * 4;
    k_stitch_clear<<<grid, 256, 0, s->stream>>>(s->stitch);
    k_stitch_insert<<<grid, 256, 0, s->stream>>>(s->stitch, gathered, s->L, nranks);
    k_stitch_union<<<grid, 256, 0, s->stream>>>(s->stitch, gathered, s->L, nranks);
    k_stitch_apply<<<(2 * s->L + 255) / 256, 256, 0, s->stream>>>(s->stitch, gathered, s->L, rank, s->y_off, s->N,
                                                                 static_cast<uint32_t *>(s->labels()), s->xroot(),
                                                                 &s->ctl()->stitch_bad);
    s->ker.flip_slab(s->pending, s->stream);
    CUDA_TRY(cudaGetLastError());
    s->launches += 5;
    s->slab_labelled = false;
    s->T += 1;
    if (s->T - s->oldest_T >= kRingCap) s->oldest_T = s->T - kRingCap + 1;
    s->have_sweep = true;
    s->labels_flat = false;
    return XY_OK;
}

int xy_debug_philox(const uint32_t *ctr, const uint32_t *key, uint32_t *out, size_t n)
{
    return debug_philox_common(ctr, key, out, n, false);
}

int xy_debug_curand_philox(const uint32_t *ctr, const uint32_t *key, uint32_t *out, size_t n)
{
    return debug_philox_common(ctr, key, out, n, true);
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------
// xy_observe_static: the observables-only pass of k_bonds for callers that must not allocate.
//
// k_bonds needs global memory beyond its input and output: one record of partial sums per CTA, the
// last-CTA ticket, and the (cos, sin)(k / 1024) table.  A state carves these out of its workspace; here
// they live in ONE file-scope device array that every GPU loading this library holds until the process
// exits (kStaticScratchBytes, about 0.4 MB).  Nothing on this path calls cudaMalloc / cudaFree or a
// library routine that allocates device memory.
// ---------------------------------------------------------------------------------------------
namespace {

constexpr size_t cx_align256(size_t v) { return (v + 255) / 256 * 256; }
constexpr size_t kStaticOffPartials = 0;
constexpr size_t kStaticOffTab = cx_align256(kStaticOffPartials + (size_t)kMaxGrid * kPartialStride * sizeof(double));
constexpr size_t kStaticOffCtl = cx_align256(kStaticOffTab + (size_t)(kTabN + 1) * sizeof(double2));
constexpr size_t kStaticScratchBytes = cx_align256(kStaticOffCtl + sizeof(DevCtl));
static_assert(kStaticScratchBytes == 406528, "include/xy.h states this size");

// In host code this name is only a handle for cudaGetSymbolAddress: it is NOT a device address.
static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];

constexpr int kStaticMaxDevices = 64;
struct StaticDev {
    bool ready = false;
    unsigned char *base = nullptr;     // device address of g_static_scratch on this device
    int sms = 0;
    int occ[2][2] = {{0, 0}, {0, 0}};  // CTAs per SM of k_bonds<VEC, RS, false, true, false>: [VEC == 4][RS == kRSLarge]
};
StaticDev g_static_dev[kStaticMaxDevices];
std::mutex g_static_mu;

// once per device, with that device current: resolve the array's device address, upload the table, opt the
// four kernel variants in to their shared memory, query their occupancy, zero the control block
int static_setup(int dev, StaticDev &d)
{
    unsigned char *p = nullptr;
    CUDA_TRY(cudaGetSymbolAddress((void **)&p, g_static_scratch));
    if (!p || ((uintptr_t)p & 255u)) return fail(XY_ERR_CUDA, "static scratch has no usable device address");
    {
        std::vector<double2> h(kTabN + 1);
        for (int k = 0; k <= kTabN; ++k) {
            const long double ang = (long double)k / 1024.0L;
            h[k].x = (double)cosl(ang);
            h[k].y = (double)sinl(ang);
        }
        CUDA_TRY(cudaMemcpy(p + kStaticOffTab, h.data(), h.size() * sizeof(double2), cudaMemcpyHostToDevice));
    }
    CUDA_TRY(cudaMemset(p + kStaticOffCtl, 0, sizeof(DevCtl)));
    CUDA_TRY((KS<2, kR, kNW, kRSSmall, uint32_t>::bonds_prepare<false, true, false>(&d.occ[0][0])));
    CUDA_TRY((KS<2, kR, kNW, kRSLarge, uint32_t>::bonds_prepare<false, true, false>(&d.occ[0][1])));
    CUDA_TRY((KS<4, kR, kNW, kRSSmall, uint32_t>::bonds_prepare<false, true, false>(&d.occ[1][0])));
    CUDA_TRY((KS<4, kR, kNW, kRSLarge, uint32_t>::bonds_prepare<false, true, false>(&d.occ[1][1])));
    CUDA_TRY(cudaDeviceGetAttribute(&d.sms, cudaDevAttrMultiProcessorCount, dev));
    for (int v = 0; v < 2; ++v)
        for (int r = 0; r < 2; ++r)
            if (d.occ[v][r] < 1) return fail(XY_ERR_CUDA, "k_bonds does not fit this GPU (was the library built for sm_100a?)");
    CUDA_TRY(cudaDeviceSynchronize());
    d.base = p;
    d.ready = true;
    return XY_OK;
}

int is_device_pointer(const void *p)
{
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, p) != cudaSuccess) { cudaGetLastError(); return 0; }
    return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

}  // namespace

extern "C" int xy_observe_static(const float *dev_theta, uint32_t L, xy_obs *dev_out, void *cuda_stream)
{
    if (!dev_theta || !dev_out) return fail(XY_ERR_ARG, "NULL argument");
    if (L > 65536)
        return fail(XY_ERR_UNSUPPORTED_L, "L=%u unsupported: xy_observe_static handles lattices up to 65536 x 65536 (a multiple of 64)", L);
    if (int rc = check_L(L)) return rc;
    if (!is_device_pointer(dev_theta) || !is_device_pointer(dev_out))
        return fail(XY_ERR_ARG, "dev_theta and dev_out must be device memory");
    int dev = -1;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kStaticMaxDevices) return fail(XY_ERR_CUDA, "device ordinal %d not supported (limit %d)", dev, kStaticMaxDevices);
    StaticDev &d = g_static_dev[dev];
    {
        std::lock_guard<std::mutex> lock(g_static_mu);
        if (!d.ready)
            if (int rc = static_setup(dev, d)) return rc;
    }
    const bool vec4 = L % 128 == 0, large = L > 4096;
    const int rs = large ? kRSLarge : kRSSmall;
    const uint32_t nstrips = (L / (vec4 ? 128u : 64u)) * (L / (uint32_t)rs);
    // the grid of a state's k_bonds with observables (create_common): same partial sums in the same order
    long need = (nstrips + BondsShape<true>::warps - 1) / BondsShape<true>::warps;
    long g = (long)d.sms * d.occ[vec4][large];
    if (g > need) g = need;
    if (g > (long)kMaxGrid) g = kMaxGrid;

    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    SweepArgs a;
    memset(&a, 0, sizeof a);
    a.theta = const_cast<float *>(dev_theta);            // the observables-only variant never writes theta
    a.partials = reinterpret_cast<double *>(d.base + kStaticOffPartials);
    a.sincos_tab = reinterpret_cast<const double2 *>(d.base + kStaticOffTab);
    a.ctl = reinterpret_cast<DevCtl *>(d.base + kStaticOffCtl);
    a.ring = dev_out;                                    // ring of one record: record t % 1 = 0 is the caller's
    a.ring_cap = 1;
    a.L = L;
    a.rows = L;
    a.obs_fill = 1;
    a.cphi = 1.0;                                        // unrotated frame (phi = 0), as xy_measure
    // what must start at zero: the last-CTA ticket (left non-zero by a launch that did not finish) and the
    // fields of the record the kernel does not write; the partial sums are overwritten before they are read
    CUDA_TRY(cudaMemsetAsync(a.ctl, 0, sizeof(DevCtl), st));
    CUDA_TRY(cudaMemsetAsync(dev_out, 0, sizeof(xy_obs), st));
    cudaError_t e;
    if (vec4) e = large ? KS<4, kR, kNW, kRSLarge, uint32_t>::bonds_launch<false, true, false>(a, (int)g, st)
                        : KS<4, kR, kNW, kRSSmall, uint32_t>::bonds_launch<false, true, false>(a, (int)g, st);
    else e = large ? KS<2, kR, kNW, kRSLarge, uint32_t>::bonds_launch<false, true, false>(a, (int)g, st)
                   : KS<2, kR, kNW, kRSSmall, uint32_t>::bonds_launch<false, true, false>(a, (int)g, st);
    CUDA_TRY(e);
    return XY_OK;
}

#include "potts_api.cuh"
