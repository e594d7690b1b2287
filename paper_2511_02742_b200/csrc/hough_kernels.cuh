// hough_kernels.cuh -- sm_100a device code of libhough (see include/hough.h).
//
// One persistent CTA processes one event at a time (one block <-> one time window):
//
//   S0  stage     fp32 (u, v) -> validity test -> fixed-point (u_q, v_q) in shared memory           (O1)
//   S1  vote      lane <-> theta column, red.shared.add on a theta-fastest tile [rho][theta-strip]   (Eq. 4.1)
//   S2  scan      threshold + strict-local-maximum test on the tile (1 theta row of halo kept)        (L94, L106)
//   S3  clusters  union-find over the "on" bins, 8-connectivity                                      (keyword L29)
//   S4  rank      radix select of the K best peaks, ordered write-back of 32-byte records
//
// The accumulator never leaves shared memory on this path; an accumulator larger than shared memory is
// processed as strips of theta rows (votes are separable per theta row).
#pragma once
#ifdef HOUGH_EMU  // host model of the CUDA execution for the CPU tests (tests/emu/cuda_emu.h); never defined in the product build
#include "cuda_emu.h"
#define HOUGH_DYNAMIC_SMEM(name_) unsigned char* name_ = cuda_emu::g_smem
#else
#include <cuda_runtime.h>
#define HOUGH_DYNAMIC_SMEM(name_) extern __shared__ __align__(1024) unsigned char name_[]
#endif
#include <stdint.h>

namespace hough {

// Per-phase SM-cycle sums (diagnostic build only: -DHOUGH_PHASE_TIMERS); read back with hough_plan_debug_counters.
#ifdef HOUGH_PHASE_TIMERS
#define HOUGH_PT(k)                                                                     \
    do {                                                                                \
        __syncthreads();                                                                \
        if (threadIdx.x == 0) { const long long now_ = clock64(); pt_acc[k] += now_ - pt_last; pt_last = now_; } \
    } while (0)
#else
#define HOUGH_PT(k) do { } while (0)
#endif

// Debug-bounds build (-DHOUGH_BOUNDS): every computed shared-memory / scratch index is range-checked before the access;
// a violation sets HOUGH_STATUS_INTERNAL (bit 2 of the status word), counts itself, records its site, and the access is
// skipped -- nothing is stored out of range and nothing traps.  HB(...) is `true` in the product build.
constexpr int kStatusInternal = 4;
#ifdef HOUGH_BOUNDS
__device__ __noinline__ bool hb_fail(int* status, int site)
{
    atomicOr(status, kStatusInternal);
    atomicAdd(status + 2, 1);           // number of violations
    atomicCAS(status + 1, 0, site);     // first site seen
    return false;
}
#define HB(P_, i_, cap_, site_) (((unsigned long long)(long long)(i_) < (unsigned long long)(long long)(cap_)) ? true : hough::hb_fail((P_).status, (site_)))
#else
#define HB(P_, i_, cap_, site_) true
#endif

constexpr int kLBits = 22;                       // linear bin index L = t * n_rho + r < 2^22
constexpr uint32_t kLMask = (1u << kLBits) - 1;  // union-find words: epoch tag (10 bits) | L
constexpr uint32_t kEpochMax = (1u << (32 - kLBits)) - 1;
constexpr int kMaxThreads = 1024;

struct DevParams {
    int n_theta, n_rho, n_bins;
    int F, H, Oq, Wq, T, K;
    float coord_max, hit_scale;
    unsigned long long r2safe;  // u_q^2 + v_q^2 <= r2safe  =>  every theta votes in range
    int safe_enabled;
    int S, n_strips, row_bytes, tile_bytes;  // strip rows, strips per event, bytes per rho row of the tile
    int HB, PCAP;                            // capacity of the staged-hit buffer / the in-smem peak list
    int max_hits_per_event;
    long long max_hits;  // the plan's hit capacity: an event that ends beyond it has bad offsets (its hits would be read out of range)
    double rho_min, d_rho;
    double theta_min, theta_span;  // theta_t = theta_min + theta_span t / n_theta
    const int* Cq;  // [n_strips * S], zero padded
    const int* Sq;
    int off_hits, off_halo, off_peaks, off_kept, off_kroot, off_hist;  // byte offsets into dynamic smem
    // per-CTA scratch slabs in global memory (L2 resident in practice)
    uint32_t* parent;   // [n_ctas][n_bins]  tagged union-find parents
    uint32_t* csize;    // [n_ctas][n_bins]  component sizes, valid at union-find roots
    uint2* onlist;      // [n_ctas][n_bins]  (L, count) of every on bin
    uint2* peaks_ovf;   // [n_ctas][n_bins / 4 + 1] peaks beyond PCAP
    uint32_t* first_rows;  // [n_ctas][2][n_rho]  counts of theta rows 0 and 1 of the event (theta_wrap only)
    int theta_wrap;     // O4 / O5 continue past the last theta row into row 0 with rho mirrored (HOUGH_FLAG_THETA_WRAP, reading B9)
    uint32_t* epoch;    // [n_ctas]
    int* status;
    unsigned int* work_counter;
    unsigned long long* phase_cycles;  // [16] diagnostic counters
    // ---- fast path (hough_fast.cuh); f_enabled == 0 when the plan cannot use it
    int f_enabled;
    int rho_shift;                   // log2(n_rho) if n_rho is a power of two, else -1
    int Mq1;                         // ceil(M) + 1 >= max over theta of sqrt(C_q^2 + S_q^2)
    int fk, fsh;                     // log2(row bytes), F - fk
    int fS, f_nstrips, f_tile_bytes; // theta rows per strip (64 G), strips per event
    int fHB, fSLCAP, fPCAP;          // capacities: staged hits, strip list, peak list
    int f_oncap;                     // on bins an event may have on the fast path (union-find parents)
    int f_off_hits, f_off_halo, f_off_ihalo, f_off_slist, f_off_peaks, f_off_pidx, f_off_parent, f_off_hist, f_off_kept;
    const int* fCq;                  // [f_nstrips * fS], zero padded
    const int* fSq;
    int* deferred;                   // [max_events] events the fast kernel left to the general kernel
    unsigned int* deferred_count;
    unsigned int* f_work_counter;
};

struct Candidate {  // mirrors hough_candidate_t
    int theta_bin, rho_bin, votes, cluster_root, cluster_nbins;
    float theta, rho;
    int reserved;
};

// S6: theta of bin t, the oracle's sequence of double operations (for the default window theta_min = 0, theta_span = pi)
__device__ __forceinline__ float theta_of_bin(const DevParams& P, int t)
{
    return (float)__dadd_rn(P.theta_min, __ddiv_rn(__dmul_rn(P.theta_span, (double)t), (double)P.n_theta));
}

__device__ __forceinline__ uint32_t smem_addr(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void red_add_shared(uint32_t addr, uint32_t v)
{
#ifdef HOUGH_EMU
    uint32_t* w = static_cast<uint32_t*>(emu_shared_ptr(addr, 4, "red.shared.add.u32 outside the CTA's shared memory"));
#ifdef HOUGH_EMU_TSAN  // race-detector build of the host model: the detector must see an atomic
    if (w) __atomic_fetch_add(w, v, __ATOMIC_RELAXED);
#else
    if (w) *w += v;  // fibers of a CTA share one OS thread and switch only at barriers and collectives
#endif
#else
    asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
#endif
}

__device__ __forceinline__ uint4 lds128(uint32_t addr)
{
    uint4 w;
#ifdef HOUGH_EMU
    const uint4* q = static_cast<const uint4*>(emu_shared_ptr(addr, 16, "ld.shared.v4.u32 outside the CTA's shared memory"));
    w = q ? *q : make_uint4(0, 0, 0, 0);
#else
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(w.x), "=r"(w.y), "=r"(w.z), "=r"(w.w) : "r"(addr));
#endif
    return w;
}

__device__ __forceinline__ uint64_t mix64(uint64_t x)
{
    uint64_t z = x + 0x9E3779B97F4A7C15ULL;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}

// ---------------------------------------------------------------- union-find on tagged words (global, L2)

__device__ __forceinline__ uint32_t uf_find(uint32_t* parent, uint32_t x, uint32_t tag)
{
    uint32_t p = __ldcg(parent + x) & kLMask;
    while (p != x) {
        uint32_t gp = __ldcg(parent + p) & kLMask;
        if (gp == p) return p;
        __stcg(parent + x, tag | gp);  // path halving; x is not a root and never becomes one again
        x = gp;
        p = __ldcg(parent + x) & kLMask;
    }
    return x;
}

__device__ __forceinline__ void uf_union(uint32_t* parent, uint32_t a, uint32_t b, uint32_t tag)
{
    while (true) {
        a = uf_find(parent, a, tag);
        b = uf_find(parent, b, tag);
        if (a == b) return;
        if (a < b) { uint32_t t = a; a = b; b = t; }
        uint32_t old = atomicCAS(parent + a, tag | a, tag | b);  // hook the larger root under the smaller one
        if (old == (tag | a)) return;
    }
}

// ---------------------------------------------------------------- S0: staging

struct StageCtx {
    int2* hits;   // [hb]: safe hits from the front, unsafe hits from the back
    int* n_safe;  // shared counters
    int* n_unsafe;
    int hb;
    unsigned int* r2max;  // nullable: max of u_q^2 + v_q^2 over the valid hits (shared)
};

__device__ __forceinline__ void stage_one(const DevParams& P, const StageCtx& sc, float u, float v, unsigned int& r2loc)
{
    // valid <=> finite and |u|, |v| <= coord_max  (NaN fails the comparison, Inf exceeds coord_max)
    if (!(fabsf(u) <= P.coord_max) || !(fabsf(v) <= P.coord_max)) return;
    const int uq = __float2int_rn(u * P.hit_scale);  // exact product (power-of-two scale), ties to even
    const int vq = __float2int_rn(v * P.hit_scale);
    const unsigned long long r2 = (unsigned long long)((long long)uq * uq) + (unsigned long long)((long long)vq * vq);
    r2loc = max(r2loc, r2 > 0xffffffffull ? 0xffffffffu : (unsigned int)r2);
    if (P.safe_enabled && r2 <= P.r2safe) {
        const int i = atomicAdd(sc.n_safe, 1);
        if (HB(P, i, sc.hb, 100)) sc.hits[i] = make_int2(uq, vq);
    } else {
        const int i = sc.hb - 1 - atomicAdd(sc.n_unsafe, 1);
        if (HB(P, i, sc.hb, 100)) sc.hits[i] = make_int2(uq, vq);
    }
}

// Stage hits [g0, g0 + n) of the flat arrays: aligned float4 loads over the body, scalar loads at the ragged ends.
__device__ __forceinline__ void stage_hits(const DevParams& P, const StageCtx& sc, const float* __restrict__ u,
                                           const float* __restrict__ v, long long g0, int n)
{
    const long long a0 = g0 & ~3LL;
    const long long g1 = g0 + n;
    unsigned int r2loc = 0;
    for (long long i = a0 + 4LL * threadIdx.x; i < g1; i += 4LL * blockDim.x) {
        if (i >= g0 && i + 4 <= g1) {
            const float4 uu = __ldg(reinterpret_cast<const float4*>(u + i));
            const float4 vv = __ldg(reinterpret_cast<const float4*>(v + i));
            stage_one(P, sc, uu.x, vv.x, r2loc);
            stage_one(P, sc, uu.y, vv.y, r2loc);
            stage_one(P, sc, uu.z, vv.z, r2loc);
            stage_one(P, sc, uu.w, vv.w, r2loc);
        } else {
#pragma unroll
            for (int j = 0; j < 4; ++j)
                if (i + j >= g0 && i + j < g1) stage_one(P, sc, __ldg(u + i + j), __ldg(v + i + j), r2loc);
        }
    }
    if (sc.r2max && r2loc) atomicMax(sc.r2max, r2loc);
}

// ---------------------------------------------------------------- S1: voting
//
// Tile layout: counters [n_rho][S], theta fastest.  A 32-bit word column holds 4 / CW theta rows; lane l of
// every warp owns word columns l, l + 32, ... (G of them), so the 32 lanes of one red.shared hit 32 distinct
// banks and never the same address.  Hits are sliced across warps; every warp visits all G column groups.

template <int CW, int G, bool CHECK>
__device__ __forceinline__ void vote_hits(const DevParams& P, const int2* __restrict__ hits, int first, int n,
                                          uint32_t colbase, const int (&C)[G][4 / CW], const int (&Sn)[G][4 / CW],
                                          const int (&O)[G][4 / CW])
{
    constexpr int TPW = 4 / CW;  // theta rows per 32-bit word
    const int warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    const int F = P.F;
    const int rb = P.row_bytes;
    const unsigned n_rho = (unsigned)P.n_rho;
#pragma unroll 2
    for (int i = first + warp; i < first + n; i += nwarps) {
        const int2 h = hits[i];
#pragma unroll
        for (int g = 0; g < G; ++g) {
#pragma unroll
            for (int j = 0; j < TPW; ++j) {
                const int a = h.x * C[g][j] + (h.y * Sn[g][j] + (CHECK ? O[g][j] : P.Oq));
                const int r = a >> F;  // floor(a / 2^F)
                if ((!CHECK || (unsigned)r < n_rho) && HB(P, r, n_rho, 200)) {
                    const uint32_t addr = colbase + (uint32_t)(r * rb);
                    red_add_shared(addr + 128u * g, (CW == 2 && j == 1) ? 0x10000u : 1u);
                }
            }
        }
    }
}

template <int CW>
__device__ __forceinline__ uint32_t tile_get(const unsigned char* tile, int S, int r, int tl)
{
    if (CW == 2) return reinterpret_cast<const uint16_t*>(tile)[r * S + tl];
    return reinterpret_cast<const uint32_t*>(tile)[r * S + tl];
}

// Count at (strip-local theta row tl, rho bin r): rows -2 and -1 come from the saved halo of the previous strip;
// anything outside the grid counts as 0 (a neighbour outside the rectangle never beats an on bin).
template <int CW>
__device__ __forceinline__ uint32_t count_at(const DevParams& P, const unsigned char* tile, const uint32_t* halo, int tl, int r)
{
    if ((unsigned)r >= (unsigned)P.n_rho) return 0;
    if (tl >= 0) return tl < P.S ? tile_get<CW>(tile, P.S, r, tl) : 0;
    return halo[(tl + 2) * P.n_rho + r];
}

// Count of rho bin r of a theta row kept in global memory, seen from the other side of the theta seam (reading B9): the
// row is read mirrored, r -> n_rho - 1 - r.
__device__ __forceinline__ uint32_t mirrored_at(const DevParams& P, const uint32_t* row, int r)
{
    const int m = P.n_rho - 1 - r;
    return (unsigned)m < (unsigned)P.n_rho ? __ldcg(row + m) : 0u;
}

// Strict local maximum under the total order key = (count, -L): neighbours with a smaller linear index
// (previous theta row, or same row and r - 1) win ties.  seam_row0 (theta_wrap, last theta row only): the counts of theta
// row 0, which follows the last row mirrored and, having the smaller linear indices, wins ties.
template <int CW>
__device__ __forceinline__ bool is_peak(const DevParams& P, const unsigned char* tile, const uint32_t* halo, int tl, int r, uint32_t c,
                                        const uint32_t* seam_row0 = nullptr)
{
    if (count_at<CW>(P, tile, halo, tl - 1, r - 1) >= c) return false;
    if (count_at<CW>(P, tile, halo, tl - 1, r) >= c) return false;
    if (count_at<CW>(P, tile, halo, tl - 1, r + 1) >= c) return false;
    if (count_at<CW>(P, tile, halo, tl, r - 1) >= c) return false;
    if (count_at<CW>(P, tile, halo, tl, r + 1) > c) return false;
    if (seam_row0) {
        if (mirrored_at(P, seam_row0, r - 1) >= c) return false;
        if (mirrored_at(P, seam_row0, r) >= c) return false;
        if (mirrored_at(P, seam_row0, r + 1) >= c) return false;
        return true;
    }
    if (count_at<CW>(P, tile, halo, tl + 1, r - 1) > c) return false;
    if (count_at<CW>(P, tile, halo, tl + 1, r) > c) return false;
    if (count_at<CW>(P, tile, halo, tl + 1, r + 1) > c) return false;
    return true;
}

struct EventShared {  // static shared control block
    int event;
    int n_safe, n_unsafe;
    int n_on, n_peaks, n_kept;
    uint32_t diff_lo, diff_hi;
    int sel_bucket, sel_before;
    unsigned long long digest;
};

// ---------------------------------------------------------------- the event kernel

template <int CW, int G, bool DUMP>
__global__ void __launch_bounds__(kMaxThreads, 1)
hough_event_kernel(const DevParams P, const float* __restrict__ u, const float* __restrict__ v,
                   const long long* __restrict__ offsets, int n_events, Candidate* __restrict__ cands,
                   int* __restrict__ n_found, void* __restrict__ acc_out, int acc_is_u16,
                   unsigned long long* __restrict__ digest_out, const int* __restrict__ event_list,
                   const unsigned int* __restrict__ event_list_count)
{
    // with an event list, the kernel processes events event_list[0 .. *event_list_count) instead of 0 .. n_events
    if (event_list) n_events = (int)*event_list_count;
    constexpr int TPW = 4 / CW;
    HOUGH_DYNAMIC_SMEM(smem);
    __shared__ EventShared sh;

    unsigned char* tile = smem;
    int2* hits = reinterpret_cast<int2*>(smem + P.off_hits);
    uint32_t* halo = reinterpret_cast<uint32_t*>(smem + P.off_halo);
    uint2* peaks_s = reinterpret_cast<uint2*>(smem + P.off_peaks);
    unsigned long long* kept = reinterpret_cast<unsigned long long*>(smem + P.off_kept);
    uint32_t* kroot = reinterpret_cast<uint32_t*>(smem + P.off_kroot);
    int* hist = reinterpret_cast<int*>(smem + P.off_hist);

    const int tid = threadIdx.x, nthr = blockDim.x, lane = tid & 31;
    const uint32_t colbase = smem_addr(tile) + 4u * lane;
    const StageCtx sc{hits, &sh.n_safe, &sh.n_unsafe, P.HB, nullptr};

    uint32_t* parent = P.parent + (size_t)blockIdx.x * P.n_bins;
    uint32_t* csize = P.csize + (size_t)blockIdx.x * P.n_bins;
    uint2* onlist = P.onlist + (size_t)blockIdx.x * P.n_bins;
    uint2* peaks_ovf = P.peaks_ovf + (size_t)blockIdx.x * (P.n_bins / 4 + 1);
    uint32_t* first_rows = P.first_rows + (size_t)blockIdx.x * 2 * P.n_rho;
    const bool wrap = !DUMP && P.theta_wrap;
    uint32_t epoch = DUMP ? 0 : P.epoch[blockIdx.x];
#ifdef HOUGH_PHASE_TIMERS
    long long pt_acc[12] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
    long long pt_last = clock64();
#endif

    while (true) {
        __syncthreads();  // previous event fully done (also protects sh.event)
        if (tid == 0) {
            sh.event = (int)atomicAdd(P.work_counter, 1u);
            sh.n_on = 0;
            sh.n_peaks = 0;
            sh.n_kept = 0;
            sh.diff_lo = 0;
            sh.diff_hi = 0;
            sh.digest = 0;
        }
        __syncthreads();
        if (sh.event >= n_events) break;
        const int e = event_list ? event_list[sh.event] : sh.event;

        const long long g0 = offsets[e], g1 = offsets[e + 1];
        long long ne64 = g1 - g0;
        bool skip = false;
        if (g0 < 0 || ne64 < 0 || g1 > P.max_hits) { if (tid == 0) atomicOr(P.status, 2); skip = true; }
        else if (ne64 > (long long)P.max_hits_per_event) { if (tid == 0) atomicOr(P.status, 1); skip = true; }
        const int ne = skip ? 0 : (int)ne64;
        const int n_chunks = (ne + P.HB - 1) / P.HB;

        uint32_t tag = 0;
        if (!DUMP) {
            if (epoch == kEpochMax) {  // tags would repeat: clear the slab and start over
                for (int i = tid; i < P.n_bins; i += nthr) __stcg(parent + i, 0u);
                epoch = 0;
            }
            ++epoch;
            tag = epoch << kLBits;
            for (int i = tid; i < 2 * P.n_rho; i += nthr) halo[i] = 0;
        }

        const int n_strips_e = (DUMP || ne > 0) ? P.n_strips : 0;  // an empty event has no on bins
        HOUGH_PT(0);
        for (int strip = 0; strip < n_strips_e; ++strip) {
            const int base = strip * P.S;  // first theta row of the strip
            const bool last_strip = (strip == P.n_strips - 1);
            const bool full = base + P.S <= P.n_theta;

            // zero the tile
            {
                uint4* t4 = reinterpret_cast<uint4*>(tile);
                const int n16 = P.tile_bytes >> 4;
                for (int i = tid; i < n16; i += nthr) t4[i] = make_uint4(0, 0, 0, 0);
            }
            // this thread's theta columns: table values (C = S = 0 and an offset that maps below bin 0 beyond n_theta)
            int C[G][TPW], Sn[G][TPW], O[G][TPW];
#pragma unroll
            for (int g = 0; g < G; ++g)
#pragma unroll
                for (int j = 0; j < TPW; ++j) {
                    const int tl = (g * 32 + lane) * TPW + j;
                    C[g][j] = __ldg(P.Cq + base + tl);
                    Sn[g][j] = __ldg(P.Sq + base + tl);
                    O[g][j] = (base + tl < P.n_theta) ? P.Oq : -(1 << P.F);
                }
            HOUGH_PT(1);

            for (int chunk = 0; chunk < n_chunks; ++chunk) {
                if (n_chunks > 1 || strip == 0) {
                    __syncthreads();  // previous users of the hit buffer are done
                    if (tid == 0) { sh.n_safe = 0; sh.n_unsafe = 0; }
                    __syncthreads();
                    const int cn = min(P.HB, ne - chunk * P.HB);
                    stage_hits(P, sc, u, v, g0 + (long long)chunk * P.HB, cn);
                }
                __syncthreads();  // tile zeroed, hits staged
                HOUGH_PT(2);
                const int ns = sh.n_safe, nu = sh.n_unsafe;
                if (full) vote_hits<CW, G, false>(P, hits, 0, ns, colbase, C, Sn, O);
                else vote_hits<CW, G, true>(P, hits, 0, ns, colbase, C, Sn, O);
                vote_hits<CW, G, true>(P, hits, P.HB - nu, nu, colbase, C, Sn, O);
            }
            __syncthreads();  // all votes of the strip are in
            HOUGH_PT(3);

            if (DUMP) {
                // materialise the strip: acc_out[e][t][r], theta-major; digest over non-zero bins
                const int rows = min(P.S, P.n_theta - base);
                unsigned long long dsum = 0;
                for (int i = tid; i < rows * P.n_rho; i += nthr) {
                    const int tl = i / P.n_rho, r = i - tl * P.n_rho;
                    const uint32_t c = tile_get<CW>(tile, P.S, r, tl);
                    const size_t L = (size_t)(base + tl) * P.n_rho + r;
                    if (acc_out) {
                        if (acc_is_u16) reinterpret_cast<uint16_t*>(acc_out)[(size_t)e * P.n_bins + L] = (uint16_t)c;
                        else reinterpret_cast<int*>(acc_out)[(size_t)e * P.n_bins + L] = (int)c;
                    }
                    if (c) dsum += (unsigned long long)c * mix64((uint64_t)L);
                }
                if (digest_out) {
#pragma unroll
                    for (int o = 16; o; o >>= 1) dsum += __shfl_xor_sync(0xffffffffu, dsum, o);
                    if (lane == 0 && dsum) atomicAdd(&sh.digest, dsum);
                }
                __syncthreads();  // everyone has read the tile
                continue;
            }

            // ---------------- S2: threshold + local maxima
            if (wrap && strip == 0) {  // theta rows 0 and 1 are needed again when the last theta row is known (reading B9)
                for (int r = tid; r < P.n_rho; r += nthr) {
                    __stcg(first_rows + r, tile_get<CW>(tile, P.S, r, 0));
                    __stcg(first_rows + P.n_rho + r, tile_get<CW>(tile, P.S, r, 1));
                }
                __syncthreads();  // the last theta row may be in this very strip
            }
            if (strip > 0) {  // deferred row: the last theta row of the previous strip, now that row 0 is known
                for (int r = tid; r < P.n_rho; r += nthr) {
                    const uint32_t c = halo[P.n_rho + r];
                    if (c >= (uint32_t)P.T && is_peak<CW>(P, tile, halo, -1, r, c)) {
                        const int i = atomicAdd(&sh.n_peaks, 1);
                        const uint2 rec = make_uint2((uint32_t)((base - 1) * P.n_rho + r), c);
                        if (i < P.PCAP) peaks_s[i] = rec; else __stcg(peaks_ovf + (i - P.PCAP), rec);
                    }
                }
            }
            {
                const int cpr = P.row_bytes >> 4;  // 16-byte chunks per rho row
                const int total = P.n_rho * cpr;
                const uint4* t4 = reinterpret_cast<const uint4*>(tile);
                const uint32_t T = (uint32_t)P.T;
                const uint32_t TT = T | (T << 16);
                for (int idx = tid; idx < total; idx += nthr) {
                    const uint4 w = t4[idx];
                    const uint32_t ws[4] = {w.x, w.y, w.z, w.w};
                    if (CW == 2) {
                        if (((__vcmpgeu2(w.x, TT) | __vcmpgeu2(w.y, TT)) | (__vcmpgeu2(w.z, TT) | __vcmpgeu2(w.w, TT))) == 0) continue;
                    } else {
                        if (w.x < T && w.y < T && w.z < T && w.w < T) continue;
                    }
                    const int r = idx / cpr, q = idx - r * cpr;
#pragma unroll
                    for (int k = 0; k < 4 * TPW; ++k) {
                        const uint32_t c = (CW == 2) ? ((ws[k >> 1] >> (16 * (k & 1))) & 0xffffu) : ws[k];
                        if (c < T) continue;
                        const int tl = q * 4 * TPW + k;
                        const uint32_t L = (uint32_t)((base + tl) * P.n_rho + r);
                        const int io = atomicAdd(&sh.n_on, 1);
                        if (!HB(P, io, P.n_bins, 201) || !HB(P, L, P.n_bins, 202)) continue;
                        __stcg(onlist + io, make_uint2(L, c));
                        __stcg(parent + L, tag | L);
                        __stcg(csize + L, 0u);
                        // with theta_wrap, row 0 waits for the last row (tested after the strips) and the last row looks into row 0
                        const int tg = base + tl;
                        if ((tl < P.S - 1 || last_strip) && !(wrap && tg == 0) &&
                            is_peak<CW>(P, tile, halo, tl, r, c, (wrap && tg == P.n_theta - 1) ? first_rows : nullptr)) {
                            const int i = atomicAdd(&sh.n_peaks, 1);
                            const uint2 rec = make_uint2(L, c);
                            if (i < P.PCAP) peaks_s[i] = rec; else __stcg(peaks_ovf + (i - P.PCAP), rec);
                        }
                    }
                }
            }
            __syncthreads();
            HOUGH_PT(4);
            if (!last_strip) {  // keep the last two theta rows for the next strip's tests
                for (int r = tid; r < P.n_rho; r += nthr) {
                    halo[r] = tile_get<CW>(tile, P.S, r, P.S - 2);
                    halo[P.n_rho + r] = tile_get<CW>(tile, P.S, r, P.S - 1);
                }
            }
            __syncthreads();
            HOUGH_PT(5);
        }  // strips

        if (DUMP) {
            __syncthreads();
            if (digest_out && tid == 0) digest_out[e] = sh.digest;
            continue;
        }

        if (wrap && n_strips_e > 0) {
            // theta row 0 (skipped above): the row before it is the last theta row mirrored, whose bins have the larger linear
            // indices and lose ties; that row is still in the tile of the last strip
            const int tl_last = P.n_theta - 1 - (P.n_strips - 1) * P.S;
            for (int r = tid; r < P.n_rho; r += nthr) {
                const uint32_t c = __ldcg(first_rows + r);
                if (c < (uint32_t)P.T) continue;
                bool pk = true;
#pragma unroll
                for (int dr = -1; dr <= 1; ++dr) {
                    const int m = P.n_rho - 1 - (r + dr);
                    if ((unsigned)m < (unsigned)P.n_rho && tile_get<CW>(tile, P.S, m, tl_last) > c) pk = false;
                    if ((unsigned)(r + dr) < (unsigned)P.n_rho && __ldcg(first_rows + P.n_rho + r + dr) > c) pk = false;
                }
                if (r > 0 && __ldcg(first_rows + r - 1) >= c) pk = false;
                if (r + 1 < P.n_rho && __ldcg(first_rows + r + 1) > c) pk = false;
                if (pk) {
                    const int i = atomicAdd(&sh.n_peaks, 1);
                    const uint2 rec = make_uint2((uint32_t)r, c);
                    if (i < P.PCAP) peaks_s[i] = rec; else __stcg(peaks_ovf + (i - P.PCAP), rec);
                }
            }
            __syncthreads();
        }

        // ---------------- S3: connected components of the on mask (8-connectivity; across the theta seam only with theta_wrap)
        const int n_on = sh.n_on;
        const int n_pk = sh.n_peaks;
        for (int i = tid; i < n_on; i += nthr) {
            const uint32_t L = __ldcg(onlist + i).x;
            const int t = (int)(L / (uint32_t)P.n_rho), r = (int)(L - (uint32_t)t * P.n_rho);
            // the four neighbours with a smaller linear index; each adjacent pair is visited exactly once
            if (r > 0 && (__ldcg(parent + L - 1) >> kLBits) == epoch) uf_union(parent, L, L - 1, tag);
            if (t > 0) {
                const uint32_t up = L - (uint32_t)P.n_rho;
                if ((__ldcg(parent + up) >> kLBits) == epoch) uf_union(parent, L, up, tag);
                if (r > 0 && (__ldcg(parent + up - 1) >> kLBits) == epoch) uf_union(parent, L, up - 1, tag);
                if (r + 1 < P.n_rho && (__ldcg(parent + up + 1) >> kLBits) == epoch) uf_union(parent, L, up + 1, tag);
            } else if (wrap) {  // row 0 continues into the last theta row, rho mirrored; each pair across the seam is visited from here
#pragma unroll
                for (int dr = -1; dr <= 1; ++dr) {
                    const int m = P.n_rho - 1 - (r + dr);
                    if ((unsigned)m >= (unsigned)P.n_rho) continue;
                    const uint32_t nb = (uint32_t)((P.n_theta - 1) * P.n_rho + m);
                    if ((__ldcg(parent + nb) >> kLBits) == epoch) uf_union(parent, L, nb, tag);
                }
            }
        }
        __syncthreads();
        HOUGH_PT(6);
        for (int i = tid; i < n_on; i += nthr) {
            const uint32_t L = __ldcg(onlist + i).x;
            atomicAdd(csize + uf_find(parent, L, tag), 1u);
        }
        __threadfence();
        HOUGH_PT(7);

        // ---------------- S4: rank the peaks by key = (~votes, L) ascending, keep the first K
        auto peak_key = [&](int i) -> unsigned long long {
            const uint2 p = (i < P.PCAP) ? peaks_s[i] : __ldcg(peaks_ovf + (i - P.PCAP));
            return ((unsigned long long)(~p.y) << 32) | p.x;
        };
        unsigned long long kth = ~0ULL;
        if (n_pk > P.K) {
            // bytes in which the keys differ at all
            {
                const unsigned long long k0 = peak_key(0);
                unsigned long long d = 0;
                for (int i = tid; i < n_pk; i += nthr) d |= peak_key(i) ^ k0;
#pragma unroll
                for (int o = 16; o; o >>= 1) d |= __shfl_xor_sync(0xffffffffu, d, o);
                if (lane == 0 && d) { atomicOr(&sh.diff_lo, (uint32_t)d); atomicOr(&sh.diff_hi, (uint32_t)(d >> 32)); }
                __syncthreads();
                const unsigned long long diff = ((unsigned long long)sh.diff_hi << 32) | sh.diff_lo;
                unsigned long long prefix = 0, pmask = 0;
                int need = P.K;  // the need-th smallest key among those matching the prefix
                for (int byte = 7; byte >= 0; --byte) {
                    if (((diff >> (8 * byte)) & 0xffULL) == 0) continue;  // uniform
                    for (int i = tid; i < 256; i += nthr) hist[i] = 0;
                    __syncthreads();
                    for (int i = tid; i < n_pk; i += nthr) {
                        const unsigned long long k = peak_key(i);
                        if ((k & pmask) == prefix) atomicAdd(&hist[(int)((k >> (8 * byte)) & 0xffULL)], 1);
                    }
                    __syncthreads();
                    if (tid < 32) {  // warp 0: bucket holding the need-th key
                        int loc[8], s = 0;
#pragma unroll
                        for (int j = 0; j < 8; ++j) { loc[j] = hist[tid * 8 + j]; s += loc[j]; }
                        int incl = s;
#pragma unroll
                        for (int o = 1; o < 32; o <<= 1) { const int y = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += y; }
                        int before = incl - s;
                        if (before < need && need <= incl) {
                            int j = 0;
                            while (before + loc[j] < need) { before += loc[j]; ++j; }
                            sh.sel_bucket = tid * 8 + j;
                            sh.sel_before = before;
                        }
                    }
                    __syncthreads();
                    prefix |= (unsigned long long)sh.sel_bucket << (8 * byte);
                    pmask |= 0xffULL << (8 * byte);
                    need -= sh.sel_before;
                    __syncthreads();
                }
                kth = prefix | (k0 & ~pmask);
            }
        } else {
            __syncthreads();
        }
        HOUGH_PT(8);
        for (int i = tid; i < n_pk; i += nthr) {
            const unsigned long long k = peak_key(i);
            if (k <= kth) { const int ik = atomicAdd(&sh.n_kept, 1); if (HB(P, ik, P.K, 203)) kept[ik] = k; }
        }
        __syncthreads();  // also orders the csize atomics before the reads below
        const int n_kept = sh.n_kept;
        // slot = number of kept keys that are smaller (keys are unique)
        unsigned long long* sorted = kept + P.K;
        for (int i = tid; i < n_kept; i += nthr) {
            const unsigned long long k = kept[i];
            int s = 0;
            for (int j = 0; j < n_kept; ++j) s += (kept[j] < k);
            if (HB(P, s, P.K, 204)) sorted[s] = k;
        }
        __syncthreads();
        for (int s = tid; s < n_kept; s += nthr) kroot[s] = uf_find(parent, (uint32_t)(sorted[s] & 0xffffffffULL), tag);
        __syncthreads();
        for (int s = tid; s < n_kept; s += nthr) {
            const unsigned long long k = sorted[s];
            const uint32_t L = (uint32_t)(k & 0xffffffffULL);
            const uint32_t c = ~(uint32_t)(k >> 32);
            const uint32_t root = kroot[s];
            int rs = 0;
            while (rs < s && kroot[rs] != root) ++rs;  // best-ranked kept peak of the same component (<= s)
            Candidate cd;
            cd.theta_bin = (int)(L / (uint32_t)P.n_rho);
            cd.rho_bin = (int)(L - (uint32_t)cd.theta_bin * P.n_rho);
            cd.votes = (int)c;
            cd.cluster_root = rs;
            cd.cluster_nbins = (int)__ldcg(csize + root);
            cd.theta = theta_of_bin(P, cd.theta_bin);
            cd.rho = (float)__dadd_rn(P.rho_min, __dmul_rn((double)cd.rho_bin + 0.5, P.d_rho));
            cd.reserved = 0;
            int4* dst = reinterpret_cast<int4*>(cands + (size_t)e * P.K + s);
            dst[0] = make_int4(cd.theta_bin, cd.rho_bin, cd.votes, cd.cluster_root);
            dst[1] = make_int4(cd.cluster_nbins, __float_as_int(cd.theta), __float_as_int(cd.rho), 0);
        }
        if (tid == 0) n_found[e] = n_pk;
        HOUGH_PT(9);
    }
    if (!DUMP && threadIdx.x == 0) P.epoch[blockIdx.x] = epoch;
#ifdef HOUGH_PHASE_TIMERS
    if (threadIdx.x == 0)
        for (int k = 0; k < 12; ++k) atomicAdd(P.phase_cycles + k, (unsigned long long)pt_acc[k]);
#endif
}

// ---------------------------------------------------------------- S5: assignment
//
// One CTA per event at a time; the event's kept candidates become (C_q[t_s], S_q[t_s], O_q - r_s 2^F - 2^(F-1))
// triples in shared memory; each thread owns hits and scans the triples (warp-uniform broadcast reads).

// KEYED: the running arg-min is one packed key per hit, key = min(|e|, W_q + 1) * 2^kbits + slot with 2^kbits >= K, so that
// "smaller |e|, then lower slot" is a single unsigned minimum (IABS + VIMNMX + VIADDMNMX on sm_100a: three ALU-pipe
// instructions per residual instead of four); the host picks it when (W_q + 2) * 2^kbits fits 32 bits.
template <bool KEYED>
__global__ void __launch_bounds__(256)
hough_assign_kernel(const DevParams P, const float* __restrict__ u, const float* __restrict__ v,
                    const long long* __restrict__ offsets, int n_events, const Candidate* __restrict__ cands,
                    const int* __restrict__ n_found, int* __restrict__ labels, int kbits, unsigned key_mul)
{
    HOUGH_DYNAMIC_SMEM(smem);
    int4* trip = reinterpret_cast<int4*>(smem);  // [K]
    const int tid = threadIdx.x, nthr = blockDim.x;
    for (int e = blockIdx.x; e < n_events; e += gridDim.x) {
        const long long g0 = offsets[e], g1 = offsets[e + 1];
        if (g0 < 0 || g1 < g0 || g1 > P.max_hits) continue;  // flagged by the find kernel
        const bool too_long = (g1 - g0) > (long long)P.max_hits_per_event;
        const int nk = too_long ? 0 : min(n_found[e], P.K);
        __syncthreads();
        for (int s = tid; s < nk; s += nthr) {
            const Candidate* c = cands + (size_t)e * P.K + s;
            const int t = c->theta_bin, r = c->rho_bin;
            const int half = P.F >= 1 ? (1 << (P.F - 1)) : 0;
            // records are caller data: one that names no bin of this plan (not written by hough_find_clusters of the same plan)
            // must not index the tables; it becomes a line no hit can reach (e = 2^31 - 1 > W_q for every hit)
            const bool in_grid = (unsigned)t < (unsigned)P.n_theta && (unsigned)r < (unsigned)P.n_rho;
            trip[s] = in_grid ? make_int4(__ldg(P.Cq + t), __ldg(P.Sq + t), P.Oq - (r << P.F) - half, s) : make_int4(0, 0, 0x7fffffff, s);
        }
        __syncthreads();
        // HPT hits per thread and trip: one broadcast load of a candidate triple serves HPT residuals.  best starts at
        // W_q + 1, so "|e| < best" alone is the eligibility test and the strict compare keeps the lowest slot on ties.
        constexpr int HPT = 4;
        const unsigned best0 = (unsigned)P.Wq + 1u;
        for (long long i0 = g0 + tid; i0 < g1; i0 += (long long)HPT * nthr) {
            int uq[HPT], vq[HPT], label[HPT];
            unsigned best[HPT];
            bool ok[HPT];
#pragma unroll
            for (int j = 0; j < HPT; ++j) {
                const long long i = i0 + (long long)j * nthr;
                float uf = 0.f, vf = 0.f;
                if (i < g1) { uf = __ldg(u + i); vf = __ldg(v + i); }
                ok[j] = (fabsf(uf) <= P.coord_max) && (fabsf(vf) <= P.coord_max);  // false for NaN
                uq[j] = ok[j] ? __float2int_rn(uf * P.hit_scale) : 0;
                vq[j] = ok[j] ? __float2int_rn(vf * P.hit_scale) : 0;
                best[j] = best0;
                label[j] = -1;
            }
            if (KEYED) {
                // best0 = W_q + 1: an ineligible residual.  key_mul = 2^kbits arrives as a kernel parameter so that the key is
                // ONE IMAD (multiply-add on the FMA pipe) and not a shift + add on the ALU pipe, which binds this loop
                const unsigned clampv = best0, mul = key_mul;
#pragma unroll
                for (int j = 0; j < HPT; ++j) best[j] = 0xffffffffu;
#pragma unroll 2
                for (int s = 0; s < nk; ++s) {
                    const int4 c = trip[s];
#pragma unroll
                    for (int j = 0; j < HPT; ++j) {
                        const int ev = uq[j] * c.x + (vq[j] * c.y + c.z);
                        const unsigned ae = min((unsigned)abs(ev), clampv);
                        best[j] = min(best[j], ae * mul + (unsigned)c.w);
                    }
                }
#pragma unroll
                for (int j = 0; j < HPT; ++j) label[j] = (best[j] >> kbits) < clampv ? (int)(best[j] & (mul - 1u)) : -1;
            } else {
#pragma unroll 2
                for (int s = 0; s < nk; ++s) {
                    const int4 c = trip[s];
#pragma unroll
                    for (int j = 0; j < HPT; ++j) {
                        const int ev = uq[j] * c.x + (vq[j] * c.y + c.z);
                        const unsigned ae = (unsigned)abs(ev);
                        if (ae < best[j]) { best[j] = ae; label[j] = s; }
                    }
                }
            }
#pragma unroll
            for (int j = 0; j < HPT; ++j) {
                const long long i = i0 + (long long)j * nthr;
                if (i < g1) labels[i] = ok[j] ? label[j] : -1;
            }
        }
    }
}

// ---------------------------------------------------------------- roofline denominator probe

// Conflict-free shared-memory atomic adds and nothing else: lane = bank, 16 fixed addresses per thread in registers
// (rows differ per thread), alternating the two increments the vote kernel uses (+1 -> ATOMS.POPC.INC, +0x10000 -> ATOMS.ADD).
__global__ void __launch_bounds__(1024, 1)
smem_atomic_peak_kernel(int iters, int rows, unsigned long long* cycles, uint32_t* sink)
{
    HOUGH_DYNAMIC_SMEM(smem);
    uint32_t* w = reinterpret_cast<uint32_t*>(smem);
    const int lane = threadIdx.x & 31;
    for (int i = threadIdx.x; i < rows * 32; i += blockDim.x) w[i] = 0;
    __syncthreads();
    const uint32_t base = smem_addr(w);
    uint32_t x = (blockIdx.x * 1315423911u) ^ (threadIdx.x * 2654435761u) ^ 0x9E3779B9u;
    uint32_t a[16];
#pragma unroll
    for (int j = 0; j < 16; ++j) {
        x = x * 1664525u + 1013904223u;
        a[j] = base + (((x >> 8) % (uint32_t)rows) * 32u + lane) * 4u;
    }
    const long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int j = 0; j < 16; ++j) red_add_shared(a[j], (j & 1) ? 0x10000u : 1u);
    }
    const long long t1 = clock64();
    __syncthreads();
    if (threadIdx.x == 0) cycles[blockIdx.x] = (unsigned long long)(t1 - t0);
    uint32_t s = 0;
    for (int i = threadIdx.x; i < rows * 32; i += blockDim.x) s += w[i];
    if (s == 0xdeadbeefu) sink[0] = s;
}

}  // namespace hough
