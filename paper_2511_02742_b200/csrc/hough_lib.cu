// hough_lib.cu -- host side of libhough: the C ABI of include/hough.h over the kernels of hough_kernels.cuh.
//
// No torch, no Python: plain CUDA runtime.  Built for sm_100a only (see paper_2511_02742_b200/build.py).
#include "../../include/hough.h"
#include "hough_kernels.cuh"
#include "hough_fast.cuh"
#include "hough_track.cuh"

#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <new>
#include <vector>

using hough::Candidate;
using hough::DevParams;

static_assert(sizeof(hough_candidate_t) == 32, "record layout");
static_assert(sizeof(Candidate) == sizeof(hough_candidate_t), "device record mirrors the ABI record");
static_assert(sizeof(hough_fit_t) == 32 && sizeof(hough::Fit) == sizeof(hough_fit_t), "fit record layout");
static_assert(sizeof(hough::FitAcc) == 48, "per-candidate accumulator");

// kernel launch: the <<< >>> syntax, or the host model of tests/emu when the sources are compiled for the CPU tests
#ifdef HOUGH_EMU
#define HOUGH_LAUNCH(kernel_, grid_, block_, smem_, stream_, ...) \
    cuda_emu::launch(dim3(grid_), dim3(block_), (size_t)(smem_), [&]() { kernel_(__VA_ARGS__); })
#else
#define HOUGH_LAUNCH(kernel_, grid_, block_, smem_, stream_, ...) kernel_<<<(grid_), (block_), (smem_), (stream_)>>>(__VA_ARGS__)
#endif

static thread_local char g_cuda_err[256] = "";

static int cuda_fail(cudaError_t e, const char* what)
{
    snprintf(g_cuda_err, sizeof g_cuda_err, "%s: %s", what, cudaGetErrorString(e));
    (void)cudaGetLastError();
    return HOUGH_ECUDA;
}
#define HCK(call)                                                   \
    do {                                                            \
        cudaError_t e_ = (call);                                    \
        if (e_ != cudaSuccess) return cuda_fail(e_, #call);         \
    } while (0)

static const int kHostChunksMax = 32;

struct hough_plan {
    hough_plan_desc_t desc;
    DevParams P;
    hough_plan_info_t info;
    std::vector<int32_t> h_cos, h_sin;
    int cw, G;  // counter bytes, column groups per tile
    int n_ctas, threads, smem_bytes;
    int assign_ctas;
    int64_t launches;
    // fast path (hough_fast.cuh)
    int f_G, f_maxt, f_minb, f_threads, f_ctas, f_smem;
    int* d_fcos;
    int* d_fsin;
    int* d_deferred;
    // owned device memory
    int* d_cos;
    int* d_sin;
    void* d_scratch;
    int* d_status;
    unsigned int* d_counter;
    // lazily created resources of hough_run_host
    bool h_ready;                        // every resource below exists
    cudaStream_t h_stream;               // compute stream of hough_run_host
    cudaStream_t h_up, h_down;           // copy streams: host -> device, device -> host
    cudaEvent_t h_ev_up[kHostChunksMax], h_ev_done[kHostChunksMax];
    float* hd_u;
    float* hd_v;
    long long* hd_off;
    Candidate* hd_cands;
    int* hd_nfound;
    int* hd_labels;
};

// Experiment switches exist only in the tuning build (-DHOUGH_TUNING, used from _work/): the results and the launch
// shape of the product library never depend on the environment of the calling process.
#ifdef HOUGH_TUNING
static int env_int(const char* name, int dflt)
{
    const char* s = getenv(name);
    return (s && *s) ? atoi(s) : dflt;
}
#else
static inline int env_int(const char*, int dflt) { return dflt; }
#endif

static size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// Shared-memory footprint of everything but the tile.
struct SmemLayout {
    int off_hits, off_halo, off_peaks, off_kept, off_kroot, off_hist, total;
};
static SmemLayout layout_smem(int tile_bytes, int HB, int n_rho, int PCAP, int K)
{
    SmemLayout L;
    size_t o = align_up((size_t)tile_bytes, 1024);
    L.off_hits = (int)o;   o = align_up(o + (size_t)HB * 8, 16);
    L.off_halo = (int)o;   o = align_up(o + (size_t)2 * n_rho * 4, 16);
    L.off_peaks = (int)o;  o = align_up(o + (size_t)PCAP * 8, 16);
    L.off_kept = (int)o;   o = align_up(o + (size_t)2 * K * 8, 16);
    L.off_kroot = (int)o;  o = align_up(o + (size_t)K * 4, 16);
    L.off_hist = (int)o;   o = align_up(o + 256 * 4, 16);
    L.total = (int)o;
    return L;
}

template <int CW, int G, bool DUMP>
static cudaError_t launch_event_kernel(const hough_plan* p, const float* u, const float* v, const long long* off, int n_events,
                                       Candidate* cands, int* n_found, void* acc, int acc_u16, unsigned long long* digest,
                                       cudaStream_t st, const int* elist, const unsigned int* ecount)
{
    auto k = hough::hough_event_kernel<CW, G, DUMP>;
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, p->smem_bytes);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(k, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    if (e != cudaSuccess) return e;
    HOUGH_LAUNCH(k, p->n_ctas, p->threads, p->smem_bytes, st, p->P, u, v, off, n_events, cands, n_found, acc, acc_u16, digest, elist, ecount);
    return cudaGetLastError();
}

template <bool DUMP>
static cudaError_t dispatch_event_kernel(const hough_plan* p, const float* u, const float* v, const long long* off, int n_events,
                                         Candidate* cands, int* n_found, void* acc, int acc_u16, unsigned long long* digest,
                                         cudaStream_t st, const int* elist = nullptr, const unsigned int* ecount = nullptr)
{
#define HOUGH_CASE(CW_, G_)                                                                                                 \
    if (p->cw == CW_ && p->G == G_)                                                                                         \
        return launch_event_kernel<CW_, G_, DUMP>(p, u, v, off, n_events, cands, n_found, acc, acc_u16, digest, st, elist, ecount);
    HOUGH_CASE(2, 1) HOUGH_CASE(2, 2) HOUGH_CASE(2, 3) HOUGH_CASE(2, 4) HOUGH_CASE(2, 6) HOUGH_CASE(2, 8)
    HOUGH_CASE(4, 1) HOUGH_CASE(4, 2) HOUGH_CASE(4, 3) HOUGH_CASE(4, 4) HOUGH_CASE(4, 6) HOUGH_CASE(4, 8)
#undef HOUGH_CASE
    return cudaErrorInvalidValue;
}

static const int kGroupChoices[] = {8, 6, 4, 3, 2, 1};

// ---- fast kernel: instantiations (G, max threads, min CTAs per SM) and their launch
template <int G, int MAXT, int MINB>
static cudaError_t launch_fast(const hough_plan* p, const float* u, const float* v, const long long* off, int n_events,
                               Candidate* cands, int* n_found, cudaStream_t st)
{
    auto k = hough::hough_fast_kernel<G, MAXT, MINB>;
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, p->f_smem);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(k, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    if (e != cudaSuccess) return e;
    HOUGH_LAUNCH(k, p->f_ctas, p->f_threads, p->f_smem, st, p->P, u, v, off, n_events, cands, n_found);
    return cudaGetLastError();
}

static cudaError_t dispatch_fast(const hough_plan* p, const float* u, const float* v, const long long* off, int n_events,
                                 Candidate* cands, int* n_found, cudaStream_t st)
{
#define HOUGH_FCASE(G_, T_, B_)                                                                   \
    if (p->f_G == G_ && p->f_maxt == T_ && p->f_minb == B_) return launch_fast<G_, T_, B_>(p, u, v, off, n_events, cands, n_found, st);
    // the shapes hough_plan_create can choose (its preference list); the tuning build adds the ones experiments asked for
    HOUGH_FCASE(1, 1024, 1) HOUGH_FCASE(2, 1024, 1) HOUGH_FCASE(4, 1024, 1)
    HOUGH_FCASE(1, 768, 2) HOUGH_FCASE(2, 768, 2) HOUGH_FCASE(4, 768, 2)
#ifdef HOUGH_TUNING
    HOUGH_FCASE(1, 1024, 2) HOUGH_FCASE(2, 1024, 2) HOUGH_FCASE(4, 1024, 2)
    HOUGH_FCASE(1, 512, 3) HOUGH_FCASE(2, 512, 3)
#endif
#undef HOUGH_FCASE
    return cudaErrorInvalidValue;
}

struct FastLayout {
    int off_hits, off_halo, off_ihalo, off_slist, off_peaks, off_pidx, off_parent, off_hist, off_kept, total;
};
static FastLayout layout_fast(int tile_bytes, int HB, int n_rho, int SLCAP, int PCAP, int ONCAP, int K)
{
    FastLayout L;
    size_t o = align_up((size_t)tile_bytes, 16);
    L.off_hits = (int)o;   o = align_up(o + (size_t)HB * 8, 16);
    L.off_halo = (int)o;   o = align_up(o + (size_t)4 * n_rho * 2, 16);
    L.off_ihalo = (int)o;  o = align_up(o + (size_t)2 * n_rho * 2, 16);
    L.off_slist = (int)o;  o = align_up(o + (size_t)SLCAP * 4, 16);
    L.off_peaks = (int)o;  o = align_up(o + (size_t)PCAP * 4, 16);
    L.off_pidx = (int)o;   o = align_up(o + (size_t)PCAP * 2, 16);
    L.off_parent = (int)o; o = align_up(o + (size_t)ONCAP * 2, 16);
    L.off_hist = (int)o;   o = align_up(o + 256 * 4, 16);
    L.off_kept = (int)o;   o = align_up(o + (size_t)K * 20, 16);
    o += 64;               // FastShared control block
    L.total = (int)o;
    return L;
}

extern "C" {

static void free_host_path(hough_plan_t* p);

int hough_version(void) { return 200; }

const char* hough_strerror(int s)
{
    switch (s) {
        case HOUGH_OK: return "ok";
        case HOUGH_EINVAL: return "invalid argument";
        case HOUGH_ERANGE: return "parameter outside the supported range (int32 proof or plan capacity)";
        case HOUGH_ECUDA: return "CUDA error";
        case HOUGH_ENOMEM: return "out of memory";
        default: return "unknown status";
    }
}

const char* hough_last_cuda_error(void) { return g_cuda_err; }

int hough_plan_create(const hough_plan_desc_t* d, hough_plan_t** out)
{
    if (!d || !out) return HOUGH_EINVAL;
    if (d->n_theta < 1 || d->n_rho < 1 || !(d->rho_max > d->rho_min) || !isfinite(d->rho_min) || !isfinite(d->rho_max)) return HOUGH_EINVAL;
    if (!(d->coord_max > 0) || !isfinite(d->coord_max)) return HOUGH_EINVAL;
    if (d->vote_threshold < 1 || !(d->assign_window >= 0) || !isfinite(d->assign_window)) return HOUGH_EINVAL;
    if (d->max_candidates < 1 || d->max_candidates > 4096) return HOUGH_EINVAL;
    if (d->count_dtype != HOUGH_I32 && d->count_dtype != HOUGH_U16) return HOUGH_EINVAL;
    if (d->max_events < 1 || d->max_hits < 0 || d->max_hits_per_event < 0 || d->device < 0) return HOUGH_EINVAL;
    if (d->flags & ~(HOUGH_FLAG_GENERAL_ONLY | HOUGH_FLAG_SMALL_LISTS | HOUGH_FLAG_THETA_WRAP)) return HOUGH_EINVAL;
    // theta window: (0, 0) = the paper's [0, pi)
    const bool th_default = d->theta_min == 0.0 && d->theta_max == 0.0;
    const double th_lo = d->theta_min, th_hi = th_default ? 3.14159265358979323846 : d->theta_max;
    if (!isfinite(th_lo) || !isfinite(th_hi) || !(th_hi > th_lo) || th_hi - th_lo > 6.283185307179586) return HOUGH_EINVAL;
    // theta wrap (reading B9): row n_theta is row 0 with rho mirrored -- true only for [0, pi) and a rho range symmetric about 0
    const bool theta_wrap = (d->flags & HOUGH_FLAG_THETA_WRAP) != 0;
    if (theta_wrap && (!(th_default || (th_lo == 0.0 && th_hi == 3.14159265358979323846)) || d->rho_min != -d->rho_max || d->n_theta < 3))
        return HOUGH_EINVAL;
    if (d->count_dtype == HOUGH_U16 && d->max_hits_per_event > 65535) return HOUGH_ERANGE;  // a bin gets <= 1 vote per hit
    if ((int64_t)d->n_theta * d->n_rho > (1ll << hough::kLBits)) return HOUGH_ERANGE;
    const int H = d->hit_frac_bits < 0 ? 6 : d->hit_frac_bits;
    if (H > 20) return HOUGH_ERANGE;

    // ---- fixed-point constants (host double precision, llround = half away from zero)
    const double d_rho = (d->rho_max - d->rho_min) / d->n_rho;
    // int32 proof of a given F: |u_q C| + |v_q S| + |O_q| <= 2^31 - 1 for every valid hit (|u_q|, |v_q| <= q_max = floor(coord_max 2^H
    // + 1/2); the corner hits attain q_max (|C| + |S|)), and the bin centres r 2^F + 2^(F-1) of the assignment fit too
    auto int32_proof = [&](int f) {
        const double m = ldexp(1.0, f - H) / d_rho;
        double max_cs = 0.0;
        for (int t = 0; t < d->n_theta; ++t) {
            const double th = th_lo + (th_hi - th_lo) * t / d->n_theta;
            const double cs = fabs((double)llround(cos(th) * m)) + fabs((double)llround(sin(th) * m));
            if (cs > max_cs) max_cs = cs;
        }
        const double qmax = floor(d->coord_max * ldexp(1.0, H) + 0.5);
        const double oq = fabs((double)llround(-d->rho_min * ldexp(1.0, f) / d_rho));
        return qmax * max_cs + oq <= 2147483647.0 && ((double)d->n_rho + 1.0) * ldexp(1.0, f) <= 2147483647.0;
    };
    int F = d->acc_frac_bits;
    if (F < 0) {  // the largest F <= 24 that passes the proof: closed form first (O2), then down until it holds
        const double amin = fabs(d->rho_min), amax = fabs(d->rho_max);
        double span = sqrt(2.0) * d->coord_max / d_rho + (amin > amax ? amin : amax) / d_rho + 2.0;
        if (span < (double)d->n_rho + 1.0) span = (double)d->n_rho + 1.0;
        F = 24;
        while (F > 0 && span * ldexp(1.0, F) > 2147483647.0) --F;
        while (F > 1 && !int32_proof(F)) --F;
    }
    if (F > 30 || F < 1) return HOUGH_ERANGE;
    if (fabs(d->rho_min) * ldexp(1.0, F) / d_rho > 2147483646.0 || !int32_proof(F)) return HOUGH_ERANGE;
    const double M = ldexp(1.0, F - H) / d_rho;
    const double oq_d = -d->rho_min * ldexp(1.0, F) / d_rho;
    const double wq_d = d->assign_window * ldexp(1.0, F) / d_rho;
    if (fabs(oq_d) > 2147483646.0 || wq_d > 2147483646.0 || M > 2147483646.0) return HOUGH_ERANGE;
    const long long Oq = llround(oq_d), Wq = llround(wq_d);

    hough_plan* p = new (std::nothrow) hough_plan();
    if (!p) return HOUGH_ENOMEM;
    p->desc = *d;
    p->desc.hit_frac_bits = H;
    p->desc.acc_frac_bits = F;
    p->h_cos.resize(d->n_theta);
    p->h_sin.resize(d->n_theta);
    for (int t = 0; t < d->n_theta; ++t) {
        const double th = th_lo + (th_hi - th_lo) * t / d->n_theta;  // [0, pi): pi t / n_theta bit for bit
        const long long c = llround(cos(th) * M), s = llround(sin(th) * M);
        p->h_cos[t] = (int32_t)c;
        p->h_sin[t] = (int32_t)s;
    }
    const long long qmax = (long long)floor(d->coord_max * ldexp(1.0, H) + 0.5);

    // ---- launch configuration
    int dev_count = 0;
    cudaError_t ce = cudaGetDeviceCount(&dev_count);
    if (ce != cudaSuccess || d->device >= dev_count) { delete p; return ce != cudaSuccess ? cuda_fail(ce, "cudaGetDeviceCount") : HOUGH_EINVAL; }
    cudaDeviceProp prop;
    if ((ce = cudaSetDevice(d->device)) != cudaSuccess || (ce = cudaGetDeviceProperties(&prop, d->device)) != cudaSuccess) {
        delete p;
        return cuda_fail(ce, "cudaGetDeviceProperties");
    }
    const int n_sm = prop.multiProcessorCount;
    const int smem_optin = (int)prop.sharedMemPerBlockOptin;            // 227 KiB on B200
    const int smem_sm = (int)prop.sharedMemPerMultiprocessor;           // 228 KiB
    const int reserved = (int)prop.reservedSharedMemPerBlock;           // 1 KiB

    int cw = (d->max_hits_per_event <= 65535 && d->vote_threshold <= 65535) ? 2 : 4;
    const int cw_env = env_int("HOUGH_COUNTER_BYTES", 0);
    if (cw_env == 4) cw = 4;
    const int rpg = 32 * (4 / cw);  // theta rows per column group
    const int groups_all = (d->n_theta + rpg - 1) / rpg;
    const int K = d->max_candidates;
    const int HB = (int)align_up((size_t)(d->max_hits_per_event < 32 ? 32 : (d->max_hits_per_event > 4096 ? 4096 : d->max_hits_per_event)), 32);

    int ctas_per_sm = env_int("HOUGH_CTAS_PER_SM", 0);
    int threads = env_int("HOUGH_THREADS", 0);
    int G = env_int("HOUGH_GROUPS", 0);
    auto fits = [&](int g, int cps, int pcap) {
        // 256 bytes of headroom for the kernel's static shared variables
        const int budget = (cps == 1 ? smem_optin : (smem_sm / cps - reserved)) - 256;
        return layout_smem(d->n_rho * 128 * g, HB, d->n_rho, pcap, K).total <= (budget < smem_optin ? budget : smem_optin);
    };
    int g_cover = 8;  // smallest choice that covers every theta row (no point in allocating rows beyond n_theta)
    for (int g : kGroupChoices) if (g >= groups_all) g_cover = g;
    auto pick_G = [&](int cps) {
        for (int g : kGroupChoices)
            if (g <= g_cover && fits(g, cps, 512)) return g;
        return 0;
    };
    if (ctas_per_sm <= 0) {
        // default: two CTAs per SM when a tile of at least two column groups (or the whole grid) still fits, so that one
        // CTA's scan / cluster phases overlap the other's voting; otherwise one large CTA
        const int g2 = pick_G(2);
        ctas_per_sm = (g2 >= 2 || (g2 >= 1 && g2 >= groups_all)) ? 2 : 1;
    }
    if (G <= 0) G = pick_G(ctas_per_sm);
    if (G <= 0 && ctas_per_sm > 1) { ctas_per_sm = 1; G = pick_G(1); }
    if (G <= 0 || !fits(G, ctas_per_sm, 256)) { delete p; return HOUGH_ERANGE; }
    if (threads <= 0) threads = ctas_per_sm == 1 ? 1024 : 512;
    threads = threads / 32 * 32;
    if (threads < 32 || threads > hough::kMaxThreads) { delete p; return HOUGH_EINVAL; }
    int PCAP = 4096;
    while (PCAP > 256 && !fits(G, ctas_per_sm, PCAP)) PCAP -= 256;
    const int S = G * rpg;
    const int n_strips = (d->n_theta + S - 1) / S;
    const int tile_bytes = d->n_rho * 128 * G;
    const SmemLayout lay = layout_smem(tile_bytes, HB, d->n_rho, PCAP, K);

    p->cw = cw;
    p->G = G;
    p->threads = threads;
    p->smem_bytes = lay.total;
    p->n_ctas = n_sm * ctas_per_sm;
    p->assign_ctas = n_sm * 8;
    p->launches = 0;

    // ---- fast kernel configuration (hough_fast.cuh): u16 counters, tile rows of 128 G bytes
    p->f_G = 0;
    FastLayout flay{};
    int f_S = 0, f_nstrips = 0, f_tile = 0, f_HB = 0, f_SLCAP = 0, f_PCAP = 0, f_ONCAP = 0, f_k = 0;
    if (cw == 2 && d->vote_threshold <= 1023 && K <= 1000 && d->max_hits_per_event >= 1 && !env_int("HOUGH_NO_FAST", 0) &&
        !(d->flags & HOUGH_FLAG_GENERAL_ONLY) && !theta_wrap &&  // the fast kernel has no seam logic: wrap plans use the general kernel
        // the reachable-row bound of the fast kernel keeps u_q^2 + v_q^2 in 32 bits
        2.0 * (double)qmax * (double)qmax <= 4294967295.0) {
        struct Cand { int G, maxt, minb, threads, cps; };
        // preference order: one 1024-thread CTA per SM with the widest tile row that fits, then two CTAs per SM
        const Cand cands[] = {{4, 1024, 1, 1024, 1}, {2, 1024, 1, 1024, 1}, {1, 1024, 1, 1024, 1}, {4, 768, 2, 768, 2}, {2, 768, 2, 768, 2}, {1, 768, 2, 768, 2}};
        const int want_G = env_int("HOUGH_FAST_G", 0), want_t = env_int("HOUGH_FAST_MAXT", 0), want_b = env_int("HOUGH_FAST_MINB", 0);
        std::vector<Cand> list(cands, cands + sizeof(cands) / sizeof(cands[0]));
        if (want_G && want_t && want_b) list.assign(1, Cand{want_G, want_t, want_b, want_t, want_b}  /* the kernel assumes blockDim.x == MAXT */);
        for (const Cand& c : list) {
            const int rows = 64 * c.G;
            if (rows > 64 && rows / 2 >= d->n_theta) continue;  // a narrower tile already covers every theta row
            int kk = 7; while ((128 << (kk - 7)) < 128 * c.G) ++kk;
            const int sh = F - kk;
            if (sh < 0) continue;
            // unsigned range of a' = a + (tile_base << sh): tile_base < 4096 (window offset of the dynamic allocation)
            if (((unsigned long long)4096 << sh) + ((unsigned long long)d->n_rho << F) > 0xffffffffull) continue;
            const int budget = (c.cps == 1 ? smem_optin : (smem_sm / c.cps - reserved)) - 128;  // the kernel has no static shared memory
            const int lim = budget < smem_optin ? budget : smem_optin;
            const int tile = d->n_rho * 128 * c.G;
            if ((long long)d->n_rho * rows >= (1ll << 17)) continue;  // strip-list entries hold a 17-bit tile index
            int hb = (int)align_up((size_t)(d->max_hits_per_event < 32 ? 32 : d->max_hits_per_event), 32);
            if (hb > 8192) hb = 8192;
            // the strip list also holds the strip's on-chunk list at its end (hough_fast.cuh S2)
            int slcap = env_int("HOUGH_FAST_SLCAP", 2560 * c.G > 10240 ? 10240 : 2560 * c.G), pcap = env_int("HOUGH_FAST_PCAP", 3584);
            int oncap = env_int("HOUGH_FAST_ONCAP", 12288);
            if (d->flags & HOUGH_FLAG_SMALL_LISTS) { slcap = 64; pcap = 4; oncap = 16; }  // events overflow and are deferred
            if (oncap > 32767) oncap = 32767;
            if (oncap * 4 > tile) oncap = tile / 4;  // root tags reuse the tile
            auto total = [&]() { return layout_fast(tile, hb, d->n_rho, slcap, pcap, oncap, K).total; };
            while (total() > lim && pcap > 2048) pcap -= 256;
            while (total() > lim && oncap > 6144) oncap -= 512;
            while (total() > lim && slcap > 1024) slcap -= 256;
            while (total() > lim && hb > 1024) hb -= 32;
            const FastLayout L = layout_fast(tile, hb, d->n_rho, slcap, pcap, oncap, K);
            if (L.total > lim) continue;
            p->f_G = c.G; p->f_maxt = c.maxt; p->f_minb = c.minb; p->f_threads = c.threads; p->f_ctas = n_sm * c.cps; p->f_smem = L.total;
            flay = L; f_S = rows; f_nstrips = (d->n_theta + rows - 1) / rows; f_tile = tile; f_HB = hb; f_SLCAP = slcap; f_PCAP = pcap;
            f_ONCAP = oncap; f_k = kk;
            break;
        }
    }

    // ---- device memory
    const size_t n_bins = (size_t)d->n_theta * d->n_rho;
    const size_t tab = (size_t)n_strips * S;
    const size_t per_cta = n_bins * 4 + n_bins * 4 + n_bins * 8 + (n_bins / 4 + 1) * 8 + (size_t)d->n_rho * 8 + 256 + 16;
    const size_t scratch_bytes = align_up(per_cta, 256) * p->n_ctas + 256;
    std::vector<int32_t> padc(tab, 0), pads(tab, 0);
    memcpy(padc.data(), p->h_cos.data(), sizeof(int32_t) * d->n_theta);
    memcpy(pads.data(), p->h_sin.data(), sizeof(int32_t) * d->n_theta);
    bool ok = true;
    ok = ok && (ce = cudaMalloc((void**)&p->d_cos, tab * 4)) == cudaSuccess;
    ok = ok && (ce = cudaMalloc((void**)&p->d_sin, tab * 4)) == cudaSuccess;
    ok = ok && (ce = cudaMalloc(&p->d_scratch, scratch_bytes)) == cudaSuccess;
    ok = ok && (ce = cudaMalloc((void**)&p->d_status, 256)) == cudaSuccess;
    ok = ok && (ce = cudaMemcpy(p->d_cos, padc.data(), tab * 4, cudaMemcpyHostToDevice)) == cudaSuccess;
    ok = ok && (ce = cudaMemcpy(p->d_sin, pads.data(), tab * 4, cudaMemcpyHostToDevice)) == cudaSuccess;
    ok = ok && (ce = cudaMemset(p->d_scratch, 0, scratch_bytes)) == cudaSuccess;
    ok = ok && (ce = cudaMemset(p->d_status, 0, 256)) == cudaSuccess;
    const int f_oncap = f_ONCAP;
    if (p->f_G) {
        const size_t ftab = (size_t)f_nstrips * f_S;
        std::vector<int32_t> fc(ftab, 0), fs(ftab, 0);
        memcpy(fc.data(), p->h_cos.data(), sizeof(int32_t) * d->n_theta);
        memcpy(fs.data(), p->h_sin.data(), sizeof(int32_t) * d->n_theta);
        ok = ok && (ce = cudaMalloc((void**)&p->d_fcos, ftab * 4)) == cudaSuccess;
        ok = ok && (ce = cudaMalloc((void**)&p->d_fsin, ftab * 4)) == cudaSuccess;
        ok = ok && (ce = cudaMalloc((void**)&p->d_deferred, (size_t)d->max_events * 4)) == cudaSuccess;
        ok = ok && (ce = cudaMemcpy(p->d_fcos, fc.data(), ftab * 4, cudaMemcpyHostToDevice)) == cudaSuccess;
        ok = ok && (ce = cudaMemcpy(p->d_fsin, fs.data(), ftab * 4, cudaMemcpyHostToDevice)) == cudaSuccess;
    }
    if (!ok) {
        const int rc = (ce == cudaErrorMemoryAllocation) ? HOUGH_ENOMEM : cuda_fail(ce, "plan allocation");
        (void)cudaGetLastError();
        hough_plan_destroy(p);
        return rc;
    }
    p->d_counter = reinterpret_cast<unsigned int*>(p->d_status) + 16;

    DevParams& P = p->P;
    memset(&P, 0, sizeof P);
    P.n_theta = d->n_theta; P.n_rho = d->n_rho; P.n_bins = (int)n_bins;
    P.F = F; P.H = H; P.Oq = (int)Oq; P.Wq = (int)Wq; P.T = d->vote_threshold; P.K = K;
    P.coord_max = (float)d->coord_max;
    // fp32 compare |u| <= coord_max must equal the double compare of the definition: round coord_max DOWN to fp32
    if ((double)P.coord_max > d->coord_max) P.coord_max = nextafterf(P.coord_max, 0.0f);
    P.hit_scale = ldexpf(1.0f, H);
    {
        // safe radius: R (M + 1) <= min(O_q, n_rho 2^F - 1 - O_q)  =>  0 <= a < n_rho 2^F for every theta (Cauchy-Schwarz)
        const double lo = (double)Oq, hi = (double)d->n_rho * ldexp(1.0, F) - 1.0 - (double)Oq;
        const double m = lo < hi ? lo : hi;
        if (m > 0) {
            const double R = m / (M + 1.0);
            const double r2 = floor(R * R * (1.0 - 1e-9)) - 1.0;
            P.safe_enabled = r2 >= 0;
            P.r2safe = r2 >= 0 ? (unsigned long long)r2 : 0;
        }
        if (env_int("HOUGH_NO_SAFE_PATH", 0)) P.safe_enabled = 0;
    }
    P.S = S; P.n_strips = n_strips; P.row_bytes = 128 * G; P.tile_bytes = tile_bytes;
    P.HB = HB; P.PCAP = PCAP;
    P.max_hits_per_event = d->max_hits_per_event;
    P.max_hits = d->max_hits;
    P.rho_min = d->rho_min; P.d_rho = d_rho;
    P.theta_min = th_lo; P.theta_span = th_hi - th_lo;
    P.theta_wrap = theta_wrap ? 1 : 0;
    P.Cq = p->d_cos; P.Sq = p->d_sin;
    P.off_hits = lay.off_hits; P.off_halo = lay.off_halo; P.off_peaks = lay.off_peaks;
    P.off_kept = lay.off_kept; P.off_kroot = lay.off_kroot; P.off_hist = lay.off_hist;
    {
        unsigned char* b = static_cast<unsigned char*>(p->d_scratch);
        const size_t nc = (size_t)p->n_ctas;
        P.parent = reinterpret_cast<uint32_t*>(b);              b += align_up(n_bins * 4 * nc, 256);
        P.csize = reinterpret_cast<uint32_t*>(b);               b += align_up(n_bins * 4 * nc, 256);
        P.onlist = reinterpret_cast<uint2*>(b);                 b += align_up(n_bins * 8 * nc, 256);
        P.peaks_ovf = reinterpret_cast<uint2*>(b);              b += align_up((n_bins / 4 + 1) * 8 * nc, 256);
        P.first_rows = reinterpret_cast<uint32_t*>(b);          b += align_up((size_t)d->n_rho * 8 * nc, 256);
        P.epoch = reinterpret_cast<uint32_t*>(b);
        if ((size_t)(b - static_cast<unsigned char*>(p->d_scratch)) + nc * 4 > scratch_bytes) { hough_plan_destroy(p); return HOUGH_ENOMEM; }
    }
    P.status = p->d_status;
    P.work_counter = p->d_counter;
    P.f_work_counter = p->d_counter + 1;
    P.deferred_count = p->d_counter + 2;
    P.f_enabled = p->f_G != 0;
    P.Mq1 = (int)ceil(M) + 1;
    P.rho_shift = -1;
    for (int b = 0; b < 31; ++b) if ((1 << b) == d->n_rho) P.rho_shift = b;
    if (p->f_G) {
        P.fk = f_k; P.fsh = F - f_k; P.fS = f_S; P.f_nstrips = f_nstrips; P.f_tile_bytes = f_tile;
        P.fHB = f_HB; P.fSLCAP = f_SLCAP; P.fPCAP = f_PCAP; P.f_oncap = f_oncap;
        P.f_off_hits = flay.off_hits; P.f_off_halo = flay.off_halo; P.f_off_ihalo = flay.off_ihalo; P.f_off_slist = flay.off_slist;
        P.f_off_peaks = flay.off_peaks; P.f_off_pidx = flay.off_pidx; P.f_off_parent = flay.off_parent;
        P.f_off_hist = flay.off_hist; P.f_off_kept = flay.off_kept;
        P.fCq = p->d_fcos; P.fSq = p->d_fsin; P.deferred = p->d_deferred;
    }
    P.phase_cycles = reinterpret_cast<unsigned long long*>(p->d_status) + 16;  // bytes 128..255 of the status block

    hough_plan_info_t& I = p->info;
    I.hit_frac_bits = H; I.acc_frac_bits = F; I.rho_offset_q = (int32_t)Oq; I.assign_window_q = (int32_t)Wq;
    I.strip_rows = S; I.n_strips = n_strips; I.counter_bytes = cw;
    I.threads_per_cta = threads; I.ctas_per_sm = ctas_per_sm; I.n_ctas = p->n_ctas; I.smem_bytes_per_cta = lay.total;
    I.n_sm = n_sm;
    I.fast_groups = p->f_G; I.fast_threads = p->f_G ? p->f_threads : 0; I.fast_ctas = p->f_G ? p->f_ctas : 0;
    I.fast_smem_bytes = p->f_G ? p->f_smem : 0; I.fast_hits_cap = f_HB; I.fast_on_cap = f_oncap; I.fast_peak_cap = f_PCAP;
    I.fast_strip_list_cap = f_SLCAP;
    *out = p;
    return HOUGH_OK;
}

int hough_plan_destroy(hough_plan_t* p)
{
    if (!p) return HOUGH_OK;
    (void)cudaSetDevice(p->desc.device);
    (void)cudaDeviceSynchronize();
    cudaFree(p->d_cos); cudaFree(p->d_sin); cudaFree(p->d_scratch); cudaFree(p->d_status);
    cudaFree(p->d_fcos); cudaFree(p->d_fsin); cudaFree(p->d_deferred);
    free_host_path(p);
    (void)cudaGetLastError();
    delete p;
    return HOUGH_OK;
}

int hough_plan_query(const hough_plan_t* p, hough_plan_info_t* info, int32_t* h_cos_q, int32_t* h_sin_q)
{
    if (!p) return HOUGH_EINVAL;
    if (info) *info = p->info;
    if (h_cos_q) memcpy(h_cos_q, p->h_cos.data(), sizeof(int32_t) * p->h_cos.size());
    if (h_sin_q) memcpy(h_sin_q, p->h_sin.data(), sizeof(int32_t) * p->h_sin.size());
    return HOUGH_OK;
}

int64_t hough_plan_launch_count(const hough_plan_t* p) { return p ? p->launches : 0; }

int hough_plan_debug_counters(hough_plan_t* p, uint64_t* h_out16, void* stream)
{
    if (!p || !h_out16) return HOUGH_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    HCK(cudaSetDevice(p->desc.device));
    HCK(cudaMemcpyAsync(h_out16, p->P.phase_cycles, 16 * sizeof(uint64_t), cudaMemcpyDeviceToHost, st));
    HCK(cudaMemsetAsync(p->P.phase_cycles, 0, 16 * sizeof(uint64_t), st));
    unsigned int deferred = 0;  // events the last hough_find_clusters call left to the general kernel
    HCK(cudaMemcpyAsync(&deferred, p->P.deferred_count, sizeof deferred, cudaMemcpyDeviceToHost, st));
    HCK(cudaStreamSynchronize(st));
    h_out16[15] = deferred;
    int st3[3] = {0, 0, 0};  // status word, first violation site, violation count (-DHOUGH_BOUNDS build; zeros otherwise)
    HCK(cudaMemcpyAsync(st3, p->d_status, sizeof st3, cudaMemcpyDeviceToHost, st));
    HCK(cudaMemsetAsync(p->d_status + 1, 0, 2 * sizeof(int), st));
    HCK(cudaStreamSynchronize(st));
    h_out16[13] = (uint64_t)(uint32_t)st3[1];
    h_out16[14] = (uint64_t)(uint32_t)st3[2];
    return HOUGH_OK;
}

int hough_plan_status(hough_plan_t* p, int32_t* out, void* stream)
{
    if (!p || !out) return HOUGH_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    HCK(cudaSetDevice(p->desc.device));
    HCK(cudaMemcpyAsync(out, p->d_status, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    HCK(cudaMemsetAsync(p->d_status, 0, sizeof(int32_t), st));
    HCK(cudaStreamSynchronize(st));
    return HOUGH_OK;
}

static int check_common(const hough_plan_t* p, const float* u, const float* v, const int64_t* off, int32_t n_events)
{
    if (!p || !off || n_events < 0) return HOUGH_EINVAL;
    if (n_events > p->desc.max_events) return HOUGH_ERANGE;
    // u, v may be null for a batch without hits (an empty tensor has no storage); they are never read then
    if (((uintptr_t)u & 15) || ((uintptr_t)v & 15) || ((uintptr_t)off & 7)) return HOUGH_EINVAL;
    return HOUGH_OK;
}

int hough_vote(hough_plan_t* p, const float* d_u, const float* d_v, const int64_t* d_offsets, int32_t n_events, void* d_acc,
               uint64_t* d_digest, void* stream)
{
    int rc = check_common(p, d_u, d_v, d_offsets, n_events);
    if (rc) return rc;
    if (n_events == 0 || (!d_acc && !d_digest)) return HOUGH_OK;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    HCK(cudaSetDevice(p->desc.device));
    HCK(cudaMemsetAsync(p->d_counter, 0, sizeof(unsigned int), st));
    HCK(dispatch_event_kernel<true>(p, d_u, d_v, reinterpret_cast<const long long*>(d_offsets), n_events, nullptr, nullptr, d_acc,
                                    p->desc.count_dtype == HOUGH_U16, reinterpret_cast<unsigned long long*>(d_digest), st));
    p->launches += 1;
    return HOUGH_OK;
}

int hough_find_clusters(hough_plan_t* p, const float* d_u, const float* d_v, const int64_t* d_offsets, int32_t n_events,
                        hough_candidate_t* d_cands, int32_t* d_n_found, void* stream)
{
    int rc = check_common(p, d_u, d_v, d_offsets, n_events);
    if (rc) return rc;
    if (!d_cands || !d_n_found) return HOUGH_EINVAL;
    if (((uintptr_t)d_cands & 15) || ((uintptr_t)d_n_found & 3)) return HOUGH_EINVAL;
    if (n_events == 0) return HOUGH_OK;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    HCK(cudaSetDevice(p->desc.device));
    HCK(cudaMemsetAsync(p->d_counter, 0, 4 * sizeof(unsigned int), st));
    if (p->f_G) {
        // fast kernel first; the events it could not take (list in d_deferred) go through the general kernel
        HCK(dispatch_fast(p, d_u, d_v, reinterpret_cast<const long long*>(d_offsets), n_events, reinterpret_cast<Candidate*>(d_cands),
                          d_n_found, st));
        HCK(dispatch_event_kernel<false>(p, d_u, d_v, reinterpret_cast<const long long*>(d_offsets), n_events,
                                         reinterpret_cast<Candidate*>(d_cands), d_n_found, nullptr, 0, nullptr, st, p->d_deferred,
                                         p->P.deferred_count));
        p->launches += 2;
        return HOUGH_OK;
    }
    HCK(dispatch_event_kernel<false>(p, d_u, d_v, reinterpret_cast<const long long*>(d_offsets), n_events,
                                     reinterpret_cast<Candidate*>(d_cands), d_n_found, nullptr, 0, nullptr, st));
    p->launches += 1;
    return HOUGH_OK;
}

int hough_assign_hits(hough_plan_t* p, const float* d_u, const float* d_v, const int64_t* d_offsets, int32_t n_events,
                      const hough_candidate_t* d_cands, const int32_t* d_n_found, int32_t* d_labels, void* stream)
{
    int rc = check_common(p, d_u, d_v, d_offsets, n_events);
    if (rc) return rc;
    if (!d_cands || !d_n_found) return HOUGH_EINVAL;
    if (((uintptr_t)d_cands & 15) || ((uintptr_t)d_n_found & 3) || ((uintptr_t)d_labels & 3)) return HOUGH_EINVAL;
    if (n_events == 0) return HOUGH_OK;
    if (!d_labels && p->desc.max_hits > 0) return HOUGH_EINVAL;  // only a plan without hits has nothing to label
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    HCK(cudaSetDevice(p->desc.device));
    const int grid = n_events < p->assign_ctas ? n_events : p->assign_ctas;
    int kbits = 0;
    while ((1 << kbits) < p->P.K) ++kbits;
    // one packed key (|e| clamped to W_q + 1, then the slot) per hit if it fits 32 bits; else the two-register arg-min
    const bool keyed = ((unsigned long long)((unsigned)p->P.Wq + 2u) << kbits) <= 0xffffffffull;
    const size_t smem = (size_t)p->P.K * 16;
    if (keyed) {
        if (smem > 48 * 1024) HCK(cudaFuncSetAttribute(hough::hough_assign_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        HOUGH_LAUNCH(hough::hough_assign_kernel<true>, grid, 256, smem, st, p->P, d_u, d_v, reinterpret_cast<const long long*>(d_offsets),
                     n_events, reinterpret_cast<const Candidate*>(d_cands), d_n_found, d_labels, kbits, 1u << kbits);
    } else {
        if (smem > 48 * 1024) HCK(cudaFuncSetAttribute(hough::hough_assign_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        HOUGH_LAUNCH(hough::hough_assign_kernel<false>, grid, 256, smem, st, p->P, d_u, d_v, reinterpret_cast<const long long*>(d_offsets),
                     n_events, reinterpret_cast<const Candidate*>(d_cands), d_n_found, d_labels, kbits, 1u << kbits);
    }
    HCK(cudaGetLastError());
    p->launches += 1;
    return HOUGH_OK;
}

static void free_host_path(hough_plan_t* p)
{
    cudaFree(p->hd_u); cudaFree(p->hd_v); cudaFree(p->hd_off); cudaFree(p->hd_cands); cudaFree(p->hd_nfound); cudaFree(p->hd_labels);
    p->hd_u = p->hd_v = nullptr; p->hd_off = nullptr; p->hd_cands = nullptr; p->hd_nfound = p->hd_labels = nullptr;
    if (p->h_stream) cudaStreamDestroy(p->h_stream);
    if (p->h_up) cudaStreamDestroy(p->h_up);
    if (p->h_down) cudaStreamDestroy(p->h_down);
    p->h_stream = p->h_up = p->h_down = nullptr;
    for (int c = 0; c < kHostChunksMax; ++c) {
        if (p->h_ev_up[c]) cudaEventDestroy(p->h_ev_up[c]);
        if (p->h_ev_done[c]) cudaEventDestroy(p->h_ev_done[c]);
        p->h_ev_up[c] = p->h_ev_done[c] = nullptr;
    }
    p->h_ready = false;
    (void)cudaGetLastError();
}

static int init_host_path(hough_plan_t* p)
{
    const size_t mh = (size_t)(p->desc.max_hits > 0 ? p->desc.max_hits : 1) + 4, me = (size_t)p->desc.max_events;
    HCK(cudaStreamCreateWithFlags(&p->h_stream, cudaStreamNonBlocking));
    HCK(cudaStreamCreateWithFlags(&p->h_up, cudaStreamNonBlocking));
    HCK(cudaStreamCreateWithFlags(&p->h_down, cudaStreamNonBlocking));
    for (int c = 0; c < kHostChunksMax; ++c) {
        HCK(cudaEventCreateWithFlags(&p->h_ev_up[c], cudaEventDisableTiming));
        HCK(cudaEventCreateWithFlags(&p->h_ev_done[c], cudaEventDisableTiming));
    }
    HCK(cudaMalloc((void**)&p->hd_u, mh * 4));
    HCK(cudaMalloc((void**)&p->hd_v, mh * 4));
    HCK(cudaMalloc((void**)&p->hd_off, (me + 1) * 8));
    HCK(cudaMalloc((void**)&p->hd_cands, me * p->desc.max_candidates * sizeof(Candidate)));
    HCK(cudaMalloc((void**)&p->hd_nfound, me * 4));
    HCK(cudaMalloc((void**)&p->hd_labels, mh * 4));
    HCK(cudaMemset(p->hd_cands, 0, me * p->desc.max_candidates * sizeof(Candidate)));  // rows beyond n_found read as zeros
    return HOUGH_OK;
}

int hough_run_host(hough_plan_t* p, const float* h_u, const float* h_v, const int64_t* h_offsets, int32_t n_events,
                   hough_candidate_t* h_cands, int32_t* h_n_found, int32_t* h_labels)
{
    return hough_run_host_chunked(p, h_u, h_v, h_offsets, n_events, h_cands, h_n_found, h_labels, 0);
}

int hough_run_host_chunked(hough_plan_t* p, const float* h_u, const float* h_v, const int64_t* h_offsets, int32_t n_events,
                           hough_candidate_t* h_cands, int32_t* h_n_found, int32_t* h_labels, int32_t n_chunks)
{
    if (!p || !h_offsets || n_events < 0) return HOUGH_EINVAL;
    if (n_events > p->desc.max_events) return HOUGH_ERANGE;
    if (n_events == 0) return HOUGH_OK;
    if (h_offsets[0] != 0) return HOUGH_EINVAL;
    const int64_t n_hits = h_offsets[n_events];
    if (n_hits < 0 || (n_hits > 0 && (!h_u || !h_v))) return HOUGH_EINVAL;
    if (n_hits > p->desc.max_hits) return HOUGH_ERANGE;
    HCK(cudaSetDevice(p->desc.device));
    if (n_chunks < 0) return HOUGH_EINVAL;
    if (!p->h_ready) {  // lazily created; flagged ready only when every stream, event and buffer exists
        const int rc = init_host_path(p);
        if (rc != HOUGH_OK) { free_host_path(p); return rc; }
        p->h_ready = true;
    }
    // The batch is cut into chunks of events with about equal hit counts; chunk c's hits go up on one stream while chunk
    // c - 1 is computed on a second and chunk c - 2's results come down on a third (PCIe is full duplex).  The kernels of all
    // chunks run on ONE stream, in order: the plan's counters and scratch are not shared between concurrent launches.
    if (n_chunks <= 0) n_chunks = (int)(n_hits / (24ll << 20)) + 1;  // ~24 M hits (200 MB of input) per chunk
    if (n_chunks > kHostChunksMax) n_chunks = kHostChunksMax;
    if (n_chunks > n_events) n_chunks = n_events;
    const size_t K = (size_t)p->desc.max_candidates;
    cudaStream_t st = p->h_stream;
    // an error return in the middle of the batch first waits for the copies already queued: they read and write the caller's buffers
    auto drain = [&](int rc) {
        cudaStreamSynchronize(p->h_up); cudaStreamSynchronize(st); cudaStreamSynchronize(p->h_down);
        return rc;
    };
    HCK(cudaMemcpyAsync(p->hd_off, h_offsets, (size_t)(n_events + 1) * 8, cudaMemcpyHostToDevice, p->h_up));
    int e0 = 0;
    for (int c = 0; c < n_chunks; ++c) {
        int e1 = n_events;
        if (c + 1 < n_chunks) {  // first event boundary at or after the c + 1-th share of the hits
            const int64_t target = n_hits / n_chunks * (c + 1);
            int lo = e0, hi = n_events;
            while (lo < hi) { const int mid = (lo + hi) / 2; if (h_offsets[mid] < target) lo = mid + 1; else hi = mid; }
            e1 = lo < e0 ? e0 : lo;
        }
        const int ne = e1 - e0;
        const int64_t a = h_offsets[e0], z = h_offsets[e1];
        if (z < a || a < 0 || z > n_hits) return drain(HOUGH_EINVAL);  // offsets must be non-decreasing on this path
        if (z > a) {
            HCK(cudaMemcpyAsync(p->hd_u + a, h_u + a, (size_t)(z - a) * 4, cudaMemcpyHostToDevice, p->h_up));
            HCK(cudaMemcpyAsync(p->hd_v + a, h_v + a, (size_t)(z - a) * 4, cudaMemcpyHostToDevice, p->h_up));
        }
        HCK(cudaEventRecord(p->h_ev_up[c], p->h_up));
        HCK(cudaStreamWaitEvent(st, p->h_ev_up[c], 0));
        if (ne > 0) {
            int rc = hough_find_clusters(p, p->hd_u, p->hd_v, reinterpret_cast<const int64_t*>(p->hd_off) + e0, ne,
                                         reinterpret_cast<hough_candidate_t*>(p->hd_cands) + (size_t)e0 * K, p->hd_nfound + e0, st);
            if (rc) return drain(rc);
            if (h_labels) {
                rc = hough_assign_hits(p, p->hd_u, p->hd_v, reinterpret_cast<const int64_t*>(p->hd_off) + e0, ne,
                                       reinterpret_cast<const hough_candidate_t*>(p->hd_cands) + (size_t)e0 * K, p->hd_nfound + e0,
                                       p->hd_labels, st);
                if (rc) return drain(rc);
            }
        }
        HCK(cudaEventRecord(p->h_ev_done[c], st));
        HCK(cudaStreamWaitEvent(p->h_down, p->h_ev_done[c], 0));
        if (ne > 0) {
            if (h_labels && z > a) HCK(cudaMemcpyAsync(h_labels + a, p->hd_labels + a, (size_t)(z - a) * 4, cudaMemcpyDeviceToHost, p->h_down));
            if (h_cands) HCK(cudaMemcpyAsync(h_cands + (size_t)e0 * K, p->hd_cands + (size_t)e0 * K, (size_t)ne * K * sizeof(Candidate), cudaMemcpyDeviceToHost, p->h_down));
            if (h_n_found) HCK(cudaMemcpyAsync(h_n_found + e0, p->hd_nfound + e0, (size_t)ne * 4, cudaMemcpyDeviceToHost, p->h_down));
        }
        e0 = e1;
    }
    HCK(cudaStreamSynchronize(p->h_down));
    HCK(cudaStreamSynchronize(st));
    return HOUGH_OK;
}

int hough_measure_smem_atomic_peak(int32_t device, double millis, double* ops_per_s, double* sm_clock_mhz)
{
    if (!ops_per_s || device < 0 || !(millis > 0)) return HOUGH_EINVAL;
    HCK(cudaSetDevice(device));
    cudaDeviceProp prop;
    HCK(cudaGetDeviceProperties(&prop, device));
    const int threads = 1024, cps = 1, rows = 256;  // one 1024-thread CTA per SM already saturates the unit (32 lanes / clk / SM)
    const int grid = prop.multiProcessorCount * cps;
    const size_t sm = (size_t)rows * 128;
    unsigned long long* d_cyc = nullptr;
    uint32_t* d_sink = nullptr;
    HCK(cudaMalloc((void**)&d_cyc, (size_t)grid * 8));
    HCK(cudaMalloc((void**)&d_sink, 4));
    cudaEvent_t e0, e1;
    HCK(cudaEventCreate(&e0));
    HCK(cudaEventCreate(&e1));
    int iters = 2000;
    float ms = 0;
    for (int pass = 0; pass < 3; ++pass) {  // warm-up, calibration, measurement
        HCK(cudaEventRecord(e0));
        HOUGH_LAUNCH(hough::smem_atomic_peak_kernel, grid, threads, sm, (cudaStream_t)0, iters, rows, d_cyc, d_sink);
        HCK(cudaGetLastError());
        HCK(cudaEventRecord(e1));
        HCK(cudaEventSynchronize(e1));
        HCK(cudaEventElapsedTime(&ms, e0, e1));
        if (pass == 1) {
            double want = iters * (millis / (ms > 1e-3 ? ms : 1e-3));
            iters = want > 5e7 ? 50000000 : (want < 100 ? 100 : (int)want);
        }
    }
    std::vector<unsigned long long> cyc(grid);
    HCK(cudaMemcpy(cyc.data(), d_cyc, (size_t)grid * 8, cudaMemcpyDeviceToHost));
    double avg = 0;
    for (int i = 0; i < grid; ++i) avg += (double)cyc[i];
    avg /= grid;
    *ops_per_s = (double)iters * 16.0 * threads * grid / (ms * 1e-3);
    if (sm_clock_mhz) *sm_clock_mhz = avg / (ms * 1e-3) / 1e6;
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(d_cyc); cudaFree(d_sink);
    return HOUGH_OK;
}

// ---------------------------------------------------------------- back end: refit + found criterion (hough_track.cuh)

int hough_refit_tracks(hough_plan_t* p, const float* d_u, const float* d_v, const int64_t* d_offsets, int32_t n_events,
                       const int32_t* d_n_found, const int32_t* d_labels, const hough_plane_geometry_t* g, hough_fit_t* d_fits,
                       void* stream)
{
    int rc = check_common(p, d_u, d_v, d_offsets, n_events);
    if (rc) return rc;
    if (!d_n_found || !g || !d_fits || ((uintptr_t)d_fits & 15)) return HOUGH_EINVAL;
    if (g->n_planes < 1 || g->n_planes > 64 || !(g->plane_pitch > 0) || !isfinite(g->plane_pitch) || !isfinite(g->plane_origin)) return HOUGH_EINVAL;
    const int H = p->desc.hit_frac_bits;
    // exact 64-bit sums need |u_q|, |v_q| <= 2^15 and fewer than 2^16 hits per event
    if (floor(p->desc.coord_max * ldexp(1.0, H)) > 32768.0 || p->desc.max_hits_per_event > 65535) return HOUGH_ERANGE;
    const double oq_d = g->plane_origin * ldexp(1.0, H), pq_d = g->plane_pitch * ldexp(1.0, H);
    if (fabs(oq_d) > 1073741823.0 || pq_d > 1073741823.0 || llround(pq_d) < 1) return HOUGH_ERANGE;
    if (n_events == 0) return HOUGH_OK;
    if (!d_labels) return HOUGH_EINVAL;
    hough::PlaneParams G;
    G.oq = (int)llround(oq_d); G.pq = (int)llround(pq_d);
    G.n_planes = g->n_planes; G.min_run = g->min_run > 0 ? g->min_run : 5; G.wrap = g->wrap != 0;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    HCK(cudaSetDevice(p->desc.device));
    const size_t smem = (size_t)p->P.K * sizeof(hough::FitAcc);
    if (smem > 48 * 1024) HCK(cudaFuncSetAttribute(hough::hough_refit_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const int grid = n_events < p->assign_ctas ? n_events : p->assign_ctas;
    HOUGH_LAUNCH(hough::hough_refit_kernel, grid, 256, smem, st, p->P, G, d_u, d_v, reinterpret_cast<const long long*>(d_offsets), n_events,
                 d_n_found, d_labels, reinterpret_cast<hough::Fit*>(d_fits));
    HCK(cudaGetLastError());
    p->launches += 1;
    return HOUGH_OK;
}

// ---------------------------------------------------------------- variant: iterative global-maximum peel-off (hough_track.cuh)

int hough_find_tracks_peeloff(hough_plan_t* p, const float* d_u, const float* d_v, const int64_t* d_offsets, int32_t n_events,
                              hough_candidate_t* d_cands, int32_t* d_n_found, int32_t* d_labels, void* stream)
{
    int rc = check_common(p, d_u, d_v, d_offsets, n_events);
    if (rc) return rc;
    if (!d_cands || !d_n_found || ((uintptr_t)d_cands & 15) || ((uintptr_t)d_n_found & 3)) return HOUGH_EINVAL;
    if (p->desc.flags & HOUGH_FLAG_THETA_WRAP) return HOUGH_EINVAL;  // the global maximum has no neighbours to wrap
    if (n_events == 0) return HOUGH_OK;
    if (!d_labels && p->desc.max_hits > 0) return HOUGH_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    HCK(cudaSetDevice(p->desc.device));
    // theta rows per strip: as many i32 rows as fit 200 KB of shared memory
    int S = (int)((200u * 1024u) / ((size_t)p->desc.n_rho * 4));
    if (S > p->desc.n_theta) S = p->desc.n_theta;
    if (S < 1) return HOUGH_ERANGE;
    const size_t smem = (size_t)S * p->desc.n_rho * 4;
    if (smem > 48 * 1024) HCK(cudaFuncSetAttribute(hough::hough_peel_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const int grid = n_events < p->info.n_sm ? n_events : p->info.n_sm;
    HOUGH_LAUNCH(hough::hough_peel_kernel, grid, 512, smem, st, p->P, S, d_u, d_v, reinterpret_cast<const long long*>(d_offsets), n_events,
                 reinterpret_cast<Candidate*>(d_cands), d_n_found, d_labels);
    HCK(cudaGetLastError());
    p->launches += 1;
    return HOUGH_OK;
}

// ---------------------------------------------------------------- variant: two-stage (coarse -> fine) Hough (hough_track.cuh)

int hough_find_two_stage(hough_plan_t* p, const float* d_u, const float* d_v, const int64_t* d_offsets, int32_t n_events,
                         int32_t coarse_theta, int32_t coarse_rho, hough_candidate_t* d_cands, int32_t* d_n_found, void* stream)
{
    int rc = check_common(p, d_u, d_v, d_offsets, n_events);
    if (rc) return rc;
    if (!d_cands || !d_n_found || ((uintptr_t)d_cands & 15) || ((uintptr_t)d_n_found & 3)) return HOUGH_EINVAL;
    if (coarse_theta < 1 || coarse_rho < 1 || coarse_theta > p->desc.n_theta || coarse_rho > p->desc.n_rho) return HOUGH_EINVAL;
    if (p->desc.flags & HOUGH_FLAG_THETA_WRAP) return HOUGH_EINVAL;  // the coarse grid has no seam logic
    hough::TwoStageParams Q;
    Q.c_theta = coarse_theta; Q.c_rho = coarse_rho;
    Q.nT = (p->desc.n_theta + coarse_theta - 1) / coarse_theta;
    Q.nR = (p->desc.n_rho + coarse_rho - 1) / coarse_rho;
    Q.cp_cap = ((Q.nT + 1) / 2) * ((Q.nR + 1) / 2);
    size_t o = align_up((size_t)Q.nT * Q.nR * 4, 16);
    Q.off_patch = (int)o;  o = align_up(o + (size_t)9 * coarse_theta * coarse_rho * 4, 16);
    Q.off_cpeaks = (int)o; o = align_up(o + (size_t)Q.cp_cap * 8, 16);
    Q.off_ckept = (int)o;  o = align_up(o + (size_t)p->P.K * 8, 16);
    Q.off_fkeys = (int)o;  o = align_up(o + (size_t)p->P.K * 8, 16);
    if (o > 200u * 1024u) return HOUGH_ERANGE;  // the coarse histogram and its lists must fit shared memory: coarser factors
    if (n_events == 0) return HOUGH_OK;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    HCK(cudaSetDevice(p->desc.device));
    if (o > 48 * 1024) HCK(cudaFuncSetAttribute(hough::hough_two_stage_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)o));
    const int cap = p->info.n_sm * 2;
    const int grid = n_events < cap ? n_events : cap;
    HOUGH_LAUNCH(hough::hough_two_stage_kernel, grid, 512, o, st, p->P, Q, d_u, d_v, reinterpret_cast<const long long*>(d_offsets), n_events,
                 reinterpret_cast<Candidate*>(d_cands), d_n_found);
    HCK(cudaGetLastError());
    p->launches += 1;
    return HOUGH_OK;
}

// ---------------------------------------------------------------- front end: time slicing + phi (hough_track.cuh)

struct hough_frontend {
    hough_frontend_desc_t desc;
    hough::FrontParams FP;
    int n_sm;
    void* d_scratch;
};

int hough_frontend_create(const hough_frontend_desc_t* d, hough_frontend_t** out)
{
    if (!d || !out) return HOUGH_EINVAL;
    if (!(d->window_width > 0) || !(d->window_step > 0) || !isfinite(d->t0) || !isfinite(d->window_width) || !isfinite(d->window_step)) return HOUGH_EINVAL;
    if (d->windows_per_fill < 1 || d->max_fills < 1 || d->max_hits < 0 || d->device < 0 || d->reserved != 0) return HOUGH_EINVAL;
    if (!(d->xy_max > 0) || !isfinite(d->xy_max)) return HOUGH_EINVAL;
    if (d->xy_max > 512.0) return HOUGH_ERANGE;  // |x_q| <= 2^15 keeps the CORDIC state inside int32
    const double st = ldexp(1.0, hough::kTimeFracBits);
    const double t0q = d->t0 * st, sq = d->window_step * st, wq = d->window_width * st;
    if (fabs(t0q) > 1073741823.0 || sq > 1073741823.0 || wq > 1073741823.0 || llround(sq) < 1 || llround(wq) < 1) return HOUGH_ERANGE;
    if ((double)d->max_fills * d->windows_per_fill > 2147483647.0 || d->max_hits > 2147483647ll) return HOUGH_ERANGE;  // int32 src indices
    int dev_count = 0;
    cudaError_t ce = cudaGetDeviceCount(&dev_count);
    if (ce != cudaSuccess) return cuda_fail(ce, "cudaGetDeviceCount");
    if (d->device >= dev_count) return HOUGH_EINVAL;
    cudaDeviceProp prop;
    HCK(cudaSetDevice(d->device));
    HCK(cudaGetDeviceProperties(&prop, d->device));
    hough_frontend* fe = new (std::nothrow) hough_frontend();
    if (!fe) return HOUGH_ENOMEM;
    fe->desc = *d;
    fe->n_sm = prop.multiProcessorCount;
    hough::FrontParams& FP = fe->FP;
    memset(&FP, 0, sizeof FP);
    FP.t0q = (int)llround(t0q); FP.stepq = (int)llround(sq); FP.widthq = (int)llround(wq);
    FP.windows_per_fill = d->windows_per_fill;
    FP.xy_max = (float)d->xy_max;
    if ((double)FP.xy_max > d->xy_max) FP.xy_max = nextafterf(FP.xy_max, 0.0f);  // the fp32 compare must equal the double one
    for (int i = 0; i < hough::kCordicIters; ++i)
        FP.atan_q[i] = (int)llround(atan(ldexp(1.0, -i)) * (180.0 / 3.14159265358979323846) * ldexp(1.0, hough::kPhiFracBits));
    const size_t nh = (size_t)(d->max_hits > 0 ? d->max_hits : 1), nw = (size_t)d->max_fills * d->windows_per_fill;
    const size_t b_phi = align_up(nh * 4, 256), b_wr = align_up(nh * 8, 256), b_cnt = align_up(nw * 4, 256), b_cur = align_up(nw * 8, 256);
    ce = cudaMalloc(&fe->d_scratch, b_phi + b_wr + b_cnt + b_cur + 256);
    if (ce != cudaSuccess) { delete fe; (void)cudaGetLastError(); return ce == cudaErrorMemoryAllocation ? HOUGH_ENOMEM : cuda_fail(ce, "cudaMalloc"); }
    unsigned char* b = static_cast<unsigned char*>(fe->d_scratch);
    FP.wrange = reinterpret_cast<int2*>(b);           b += b_wr;
    FP.cursor = reinterpret_cast<long long*>(b);      b += b_cur;
    FP.phi = reinterpret_cast<float*>(b);             b += b_phi;
    FP.counts = reinterpret_cast<int*>(b);            b += b_cnt;
    FP.status = reinterpret_cast<int*>(b);
    ce = cudaMemset(FP.status, 0, 256);
    if (ce != cudaSuccess) { cudaFree(fe->d_scratch); delete fe; return cuda_fail(ce, "cudaMemset"); }
    *out = fe;
    return HOUGH_OK;
}

int hough_frontend_destroy(hough_frontend_t* fe)
{
    if (!fe) return HOUGH_OK;
    (void)cudaSetDevice(fe->desc.device);
    (void)cudaDeviceSynchronize();
    cudaFree(fe->d_scratch);
    (void)cudaGetLastError();
    delete fe;
    return HOUGH_OK;
}

int hough_frontend_slice(hough_frontend_t* fe, const float* d_x, const float* d_y, const float* d_z, const float* d_t,
                         const int64_t* d_fill_offsets, int32_t n_fills, int64_t n_hits, float* d_u, float* d_v, int32_t* d_src,
                         int64_t* d_offsets, int64_t capacity, void* stream)
{
    if (!fe || !d_fill_offsets || !d_offsets || n_fills < 0 || n_hits < 0 || capacity < 0) return HOUGH_EINVAL;
    if (n_fills > fe->desc.max_fills || n_hits > fe->desc.max_hits) return HOUGH_ERANGE;
    if (n_hits > 0 && (!d_x || !d_y || !d_z || !d_t)) return HOUGH_EINVAL;
    if (capacity > 0 && (!d_u || !d_v || !d_src)) return HOUGH_EINVAL;
    if (((uintptr_t)d_fill_offsets & 7) || ((uintptr_t)d_offsets & 7)) return HOUGH_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    HCK(cudaSetDevice(fe->desc.device));
    const long long nw = (long long)n_fills * fe->desc.windows_per_fill;
    if (nw == 0) { HCK(cudaMemsetAsync(d_offsets, 0, 8, st)); return HOUGH_OK; }
    HCK(cudaMemsetAsync(fe->FP.counts, 0, (size_t)nw * 4, st));
    if (n_hits > 0) {
        long long blocks = (n_hits + 255) / 256;
        const long long cap = (long long)fe->n_sm * 16;
        if (blocks > cap) blocks = cap;
        HOUGH_LAUNCH(hough::fe_count_kernel, (int)blocks, 256, 0, st, fe->FP, d_x, d_y, d_z, d_t,
                     reinterpret_cast<const long long*>(d_fill_offsets), n_fills, (long long)n_hits);
        HCK(cudaGetLastError());
    }
    HOUGH_LAUNCH(hough::fe_scan_kernel, 1, 1024, 0, st, fe->FP, nw, reinterpret_cast<long long*>(d_offsets));
    HCK(cudaGetLastError());
    if (n_hits > 0) {
        int blocks = (n_fills + 3) / 4;  // four warps per CTA, one warp per fill
        if (blocks > fe->n_sm * 16) blocks = fe->n_sm * 16;
        HOUGH_LAUNCH(hough::fe_scatter_kernel, blocks, 128, 0, st, fe->FP, d_z, reinterpret_cast<const long long*>(d_fill_offsets), n_fills,
                     (long long)n_hits, d_u, d_v, d_src, (long long)capacity);
        HCK(cudaGetLastError());
    }
    return HOUGH_OK;
}

int hough_frontend_status(hough_frontend_t* fe, int32_t* out, void* stream)
{
    if (!fe || !out) return HOUGH_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    HCK(cudaSetDevice(fe->desc.device));
    HCK(cudaMemcpyAsync(out, fe->FP.status, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    HCK(cudaMemsetAsync(fe->FP.status, 0, sizeof(int32_t), st));
    HCK(cudaStreamSynchronize(st));
    return HOUGH_OK;
}

}  // extern "C"
