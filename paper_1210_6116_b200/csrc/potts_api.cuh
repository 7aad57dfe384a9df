// potts_api.cuh -- C-ABI of the q-state Potts Swendsen-Wang sweep (include/xy.h, section "Potts").  Included at the
// end of xy_api.cu: host logic only (argument checks, workspace, launch order); the kernels are k_potts_bonds,
// k_label, k_merge (the XY sweep's, unchanged) and k_potts_flip.
#pragma once
#include "potts_kernels.cuh"

struct xy_potts {
    uint32_t L = 0, q = 0;
    uint64_t N = 0, seed = 0, T = 0;
    int device = 0;
    char *ws = nullptr;
    size_t off_labels = 0, off_bonds = 0, off_rootmask = 0, off_ctl = 0, off_stage = 0, total = 0;
    Kernels ker{};
    cudaStream_t stream = nullptr;
    bool have_sweep = false, labels_flat = false;
    double last_beta = std::numeric_limits<double>::quiet_NaN();
    unsigned long long nbx = 0, nby = 0, ncl = 0;     // of the last sweep, fetched lazily
    uint64_t launches = 0;

    uint8_t *spin() const { return reinterpret_cast<uint8_t *>(ws); }
    uint32_t *labels() const { return reinterpret_cast<uint32_t *>(ws + off_labels); }
    uint8_t *bonds() const { return reinterpret_cast<uint8_t *>(ws + off_bonds); }
    uint32_t *rootmask() const { return reinterpret_cast<uint32_t *>(ws + off_rootmask); }
    PottsCtl *ctl() const { return reinterpret_cast<PottsCtl *>(ws + off_ctl); }
    void *stage() const { return ws + off_stage; }
};

namespace {

constexpr size_t kPottsStage = 16u << 20;

SweepArgs potts_sweep_args(const xy_potts *s)
{
    SweepArgs a;
    memset(&a, 0, sizeof a);
    a.labels = s->labels();
    a.bonds = s->bonds();
    a.rootmask = s->rootmask();
    a.L = s->L;
    a.rows = s->L;
    a.tiles_x = s->L / s->ker.tw;
    a.ntiles = a.tiles_x * (s->L / s->ker.th);
    set_Ldiv(a, s->L);
    return a;
}

PottsArgs potts_args(const xy_potts *s, double beta)
{
    PottsArgs p;
    p.spin = s->spin();
    p.bonds = s->bonds();
    p.ctl = s->ctl();
    p.L = s->L;
    p.q = s->q;
    p.seed_lo = (uint32_t)(s->seed & 0xffffffffu);
    p.seed_hi = (uint32_t)(s->seed >> 32);
    p.t = (uint32_t)s->T;
    // u = (w + 0.5) 2^-32 < p  <=>  w < p 2^32 - 0.5  <=>  w < T = ceil(p 2^32 - 0.5): the scaling by 2^32 and the
    // subtraction are exact in fp64 (p 2^32 <= 2^32 has an ulp of at most 2^-20)
    const double pb = -std::expm1(-beta);
    const double x = std::ldexp(pb, 32) - 0.5;
    const double c = std::ceil(x);
    p.T = c <= 0.0 ? 0ull : (uint64_t)c;
    return p;
}

void potts_flip_launch(const xy_potts *s, const SweepArgs &a, const PottsArgs &p)
{
    if (s->ker.tw == 128) k_potts_flip<4, kR * kNW, uint32_t><<<a.ntiles, 4 * kR * kNW, 0, s->stream>>>(a, p);
    else k_potts_flip<2, kR * kNW, uint32_t><<<a.ntiles, 2 * kR * kNW, 0, s->stream>>>(a, p);
}

template <bool kB>
void potts_bonds_launch(const xy_potts *s, const PottsArgs &p)
{
    const int grid = 148 * 8;
    if (s->q <= 4) k_potts_bonds<kB, 4><<<grid, 256, 0, s->stream>>>(p);
    else if (s->q <= 8) k_potts_bonds<kB, 8><<<grid, 256, 0, s->stream>>>(p);
    else k_potts_bonds<kB, 16><<<grid, 256, 0, s->stream>>>(p);
}

}  // namespace

extern "C" {

int xy_potts_create(xy_potts **out, uint32_t L, uint32_t q, uint64_t seed, int init)
{
    if (!out) return fail(XY_ERR_ARG, "out is NULL");
    *out = nullptr;
    if (int rc = check_L(L)) return rc;
    if (q < 2 || q > (uint32_t)kPottsMaxQ) return fail(XY_ERR_ARG, "q=%u unsupported: need 2 <= q <= %d", q, kPottsMaxQ);
    if (init != XY_INIT_COLD && init != XY_INIT_HOT) return fail(XY_ERR_ARG, "init=%d unknown", init);
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0)
        return fail(XY_ERR_CUDA, "no CUDA device: this library has no CPU fallback");
    xy_potts *s = new (std::nothrow) xy_potts;
    if (!s) return fail(XY_ERR_NOMEM, "host allocation failed");
    s->L = L; s->q = q; s->N = (uint64_t)L * L; s->seed = seed;
    cudaGetDevice(&s->device);
    size_t off = align_up(s->N, 256);
    s->off_labels = off;   off = align_up(off + s->N * 4, 256);
    s->off_bonds = off;    off = align_up(off + s->N / 4, 256);
    s->off_rootmask = off; off = align_up(off + s->N / 8, 256);
    s->off_ctl = off;      off = align_up(off + sizeof(PottsCtl), 256);
    s->off_stage = off;    off = align_up(off + kPottsStage, 256);
    s->total = off;
    void *p = nullptr;
    cudaError_t e = cudaMalloc(&p, s->total);
    if (e != cudaSuccess) {
        const size_t want = s->total;
        delete s;
        cudaGetLastError();
        return fail(XY_ERR_NOMEM, "cudaMalloc(%zu) failed: %s", want, cudaGetErrorString(e));
    }
    s->ws = static_cast<char *>(p);
    s->ker = pick_kernels(L, false);
    int bo = 0, bn = 0, fl = 0;
    e = (cudaError_t)s->ker.prepare(false, &bo, &bn, &fl);
    if (e == cudaSuccess) e = cudaMemsetAsync(s->ctl(), 0, sizeof(PottsCtl), nullptr);
    if (e == cudaSuccess) {
        if (init == XY_INIT_COLD) {
            e = cudaMemsetAsync(s->spin(), 0, s->N, nullptr);
        } else {
            k_potts_init_hot<<<148 * 8, 256>>>(s->spin(), s->N, q, (uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32));
            e = cudaGetLastError();
        }
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(nullptr);
    if (e != cudaSuccess) {
        cudaFree(s->ws);
        delete s;
        return fail(XY_ERR_CUDA, "Potts state initialisation failed: %s", cudaGetErrorString(e));
    }
    *out = s;
    return XY_OK;
}

int xy_potts_destroy(xy_potts *s)
{
    if (!s) return XY_OK;
    DeviceGuard g(s->device);
    cudaStreamSynchronize(s->stream);
    cudaFree(s->ws);
    delete s;
    return XY_OK;
}

int xy_potts_sweeps(xy_potts *s, double beta, uint64_t n, void *cuda_stream)
{
    if (!s) return fail(XY_ERR_ARG, "state is NULL");
    if (!(beta >= 0.0) || !std::isfinite(beta)) return fail(XY_ERR_ARG, "beta must be finite and >= 0");
    if (s->T + n > 0xffffffffull) return fail(XY_ERR_STATE, "sweep counter would reach 2^32");
    DeviceGuard g(s->device);
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    if (st != s->stream) {
        CUDA_TRY(cudaStreamSynchronize(s->stream));
        s->stream = st;
    }
    const SweepArgs a = potts_sweep_args(s);
    for (uint64_t k = 0; k < n; ++k) {
        const PottsArgs p = potts_args(s, beta);
        CUDA_TRY(cudaMemsetAsync(s->ctl(), 0, sizeof(PottsCtl), s->stream));
        potts_bonds_launch<true>(s, p);
        s->ker.label(a, s->stream);
        s->ker.merge(a, s->stream);
        potts_flip_launch(s, a, p);
        CUDA_TRY(cudaGetLastError());
        s->launches += 4;
        s->T += 1;
    }
    if (n) { s->have_sweep = true; s->labels_flat = false; s->last_beta = beta; }
    return XY_OK;
}

int xy_potts_measure(xy_potts *s, xy_potts_obs *out)
{
    if (!s || !out) return fail(XY_ERR_ARG, "NULL argument");
    DeviceGuard g(s->device);
    PottsCtl h;
    // bond and cluster counts of the last sweep, then the link and spin counts of the CURRENT state
    CUDA_TRY(cudaMemcpyAsync(&h, s->ctl(), sizeof h, cudaMemcpyDeviceToHost, s->stream));
    CUDA_TRY(cudaStreamSynchronize(s->stream));
    const unsigned long long nbx = h.nbx, nby = h.nby, ncl = h.ncl;
    CUDA_TRY(cudaMemsetAsync(s->ctl(), 0, sizeof(PottsCtl), s->stream));
    potts_bonds_launch<false>(s, potts_args(s, 0.0));
    CUDA_TRY(cudaGetLastError());
    s->launches += 1;
    CUDA_TRY(cudaMemcpyAsync(&h, s->ctl(), sizeof h, cudaMemcpyDeviceToHost, s->stream));
    CUDA_TRY(cudaStreamSynchronize(s->stream));
    // keep the sweep's counts on the device so that a second measure returns the same record
    h.nbx = nbx; h.nby = nby; h.ncl = ncl;
    CUDA_TRY(cudaMemcpyAsync(s->ctl(), &h, sizeof h, cudaMemcpyHostToDevice, s->stream));
    CUDA_TRY(cudaStreamSynchronize(s->stream));
    memset(out, 0, sizeof *out);
    out->sweep = s->T;
    out->beta = s->last_beta;
    out->ex = h.ex; out->ey = h.ey;
    out->E = -(int64_t)(h.ex + h.ey);
    for (int k = 0; k < kPottsMaxQ; ++k) out->count[k] = h.count[k];
    out->n_bonds_x = s->have_sweep ? nbx : 0;
    out->n_bonds_y = s->have_sweep ? nby : 0;
    out->n_clusters = s->have_sweep ? ncl : 0;
    return XY_OK;
}

int xy_potts_get_spins(xy_potts *s, uint8_t *host, size_t n)
{
    if (!s || !host) return fail(XY_ERR_ARG, "NULL argument");
    if (n == 0 || n > s->N) return fail(XY_ERR_ARG, "n=%zu not in 1..L*L", n);
    DeviceGuard g(s->device);
    CUDA_TRY(cudaMemcpyAsync(host, s->spin(), n, cudaMemcpyDeviceToHost, s->stream));
    CUDA_TRY(cudaStreamSynchronize(s->stream));
    return XY_OK;
}

int xy_potts_set_spins(xy_potts *s, const uint8_t *host, size_t n)
{
    if (!s || !host) return fail(XY_ERR_ARG, "NULL argument");
    if (n != s->N) return fail(XY_ERR_ARG, "n=%zu but L*L=%llu", n, (unsigned long long)s->N);
    DeviceGuard g(s->device);
    // staged in the label array, checked there, copied to the spins only if every value is below q
    uint8_t *stage = reinterpret_cast<uint8_t *>(s->labels());
    unsigned int *flag = reinterpret_cast<unsigned int *>(s->stage());
    CUDA_TRY(cudaMemcpyAsync(stage, host, n, cudaMemcpyHostToDevice, s->stream));
    CUDA_TRY(cudaMemsetAsync(flag, 0, sizeof(unsigned int), s->stream));
    k_potts_check_spins<<<148 * 8, 256, 0, s->stream>>>(stage, s->N, s->q, flag);
    unsigned int bad = 0;
    CUDA_TRY(cudaMemcpyAsync(&bad, flag, sizeof bad, cudaMemcpyDeviceToHost, s->stream));
    CUDA_TRY(cudaStreamSynchronize(s->stream));
    s->have_sweep = false;
    if (bad) return fail(XY_ERR_ARG, "spins outside 0..q-1: rejected, the configuration is unchanged");
    CUDA_TRY(cudaMemcpyAsync(s->spin(), stage, n, cudaMemcpyDeviceToDevice, s->stream));
    CUDA_TRY(cudaMemsetAsync(s->ctl(), 0, sizeof(PottsCtl), s->stream));
    CUDA_TRY(cudaStreamSynchronize(s->stream));
    return XY_OK;
}

int xy_potts_get_sweep(xy_potts *s, uint64_t *t)
{
    if (!s || !t) return fail(XY_ERR_ARG, "NULL argument");
    *t = s->T;
    return XY_OK;
}

int xy_potts_set_sweep(xy_potts *s, uint64_t t)
{
    if (!s) return fail(XY_ERR_ARG, "state is NULL");
    if (t > 0xffffffffull) return fail(XY_ERR_STATE, "sweep counter must stay below 2^32");
    s->T = t;
    return XY_OK;
}

int xy_potts_get_bonds(xy_potts *s, uint8_t *host, size_t n)
{
    if (!s || !host) return fail(XY_ERR_ARG, "NULL argument");
    if (n == 0 || n > s->N) return fail(XY_ERR_ARG, "n=%zu not in 1..L*L", n);
    if (!s->have_sweep) return fail(XY_ERR_STATE, "no sweep has produced bonds yet");
    DeviceGuard g(s->device);
    for (uint64_t done = 0; done < n; done += kPottsStage) {
        const uint64_t m = n - done < kPottsStage ? n - done : kPottsStage;
        k_bonds_unpack<<<148 * 4, 256, 0, s->stream>>>(s->bonds(), static_cast<uint8_t *>(s->stage()), done, m);
        CUDA_TRY(cudaMemcpyAsync(host + done, s->stage(), m, cudaMemcpyDeviceToHost, s->stream));
        CUDA_TRY(cudaStreamSynchronize(s->stream));
    }
    return XY_OK;
}

int xy_potts_get_labels(xy_potts *s, int64_t *host, size_t n)
{
    if (!s || !host) return fail(XY_ERR_ARG, "NULL argument");
    if (n == 0 || n > s->N) return fail(XY_ERR_ARG, "n=%zu not in 1..L*L", n);
    if (!s->have_sweep) return fail(XY_ERR_STATE, "no sweep has produced labels yet");
    DeviceGuard g(s->device);
    if (!s->labels_flat) {
        k_flatten<uint32_t><<<148 * 8, 256, 0, s->stream>>>(s->labels(), s->N);
        CUDA_TRY(cudaGetLastError());
        s->labels_flat = true;
    }
    const uint64_t chunk = kPottsStage / sizeof(int64_t);
    for (uint64_t done = 0; done < n; done += chunk) {
        const uint64_t m = n - done < chunk ? n - done : chunk;
        k_labels_to_i64<uint32_t><<<148 * 4, 256, 0, s->stream>>>(s->labels(), static_cast<int64_t *>(s->stage()), done, m);
        CUDA_TRY(cudaMemcpyAsync(host + done, s->stage(), m * sizeof(int64_t), cudaMemcpyDeviceToHost, s->stream));
        CUDA_TRY(cudaStreamSynchronize(s->stream));
    }
    return XY_OK;
}

int xy_potts_get_launch_count(xy_potts *s, uint64_t *count)
{
    if (!s || !count) return fail(XY_ERR_ARG, "NULL argument");
    *count = s->launches;
    return XY_OK;
}

}  // extern "C"
