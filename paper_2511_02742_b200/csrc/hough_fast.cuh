// hough_fast.cuh -- the fast event kernel of libhough (sm_100a): vote + peaks + clusters with everything in shared memory.
//
// Same results as hough_event_kernel (hough_kernels.cuh), for the common case only; an event that does not fit the
// fast path's capacities is appended to a "deferred" list and processed afterwards by the general kernel:
//     more hits than the staged-hit buffer, a bin count above 1023, more peaks than the shared peak list,
//     more on bins than the cluster hash table holds, more ties at the K-th vote count than the tie buffer.
//
// Per event (one CTA at a time, several CTAs per SM so that one CTA's scan / cluster phases fill the issue slots the
// other leaves while it votes):
//   S0  stage     fp32 hits -> fixed point, "safe" hits (in range for every theta) first             (O1)
//   per strip of S = 64 G theta rows (tile [n_rho][S] of u16 counters, theta fastest, row = 128 G bytes):
//   S1  vote      lane <-> 32-bit word column (2 theta rows), 2 IMAD + SHF + LOP3 + RED per vote:
//                 the tile base is folded into the fixed-point offset, so ((a >> (F - k)) & ~(2^k - 1)) | column
//                 IS the shared-memory address of the counter word                                   (Eq. 4.1)
//   S2  scan      16-byte chunks -> compact list of on bins of the strip -> one thread per on bin:
//                 strict-local-maximum test (1 theta row of halo kept between strips)                 (L94, L106)
//   then, once per event, with the tile memory reused:
//   S4a select    vote-count histogram -> threshold count -> ties ranked by index -> K best peaks
//   S3  clusters  open-addressing hash (bin index -> slot) + union-find on the slots, 8-connectivity  (keyword L29)
//   S4b write     32-byte records in rank order
#pragma once
#include "hough_kernels.cuh"

namespace hough {

constexpr uint32_t kHashEmpty = 0xffffffffu;
constexpr int kCountBits = 10;  // packed peak key: (1023 - votes) << 22 | L   (smaller key = better rank)
constexpr uint32_t kCountMax = (1u << kCountBits) - 1;

struct FastShared {  // static shared control block
    int event;
    int n_safe, n_unsafe;
    int n_sl;     // on bins of the current strip (strip list)
    int n_on;     // on bins of the event so far (global on list)
    int n_peaks;  // peaks of the event so far
    int n_kept, n_ties;
    int defer;
    int cstar, n_gt;  // threshold vote count and number of peaks above it
};

__device__ __forceinline__ unsigned lanemask_lt()
{
    unsigned m;
    asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
    return m;
}

// Warp-aggregated append: every lane of the warp must call; returns the slot of this lane's item or -1.
__device__ __forceinline__ int warp_append(int* counter, bool pred)
{
    const unsigned m = __ballot_sync(0xffffffffu, pred);
    if (m == 0) return -1;
    const int leader = __ffs(m) - 1;
    int base = 0;
    if ((int)(threadIdx.x & 31) == leader) base = atomicAdd(counter, __popc(m));
    base = __shfl_sync(0xffffffffu, base, leader);
    return pred ? base + __popc(m & lanemask_lt()) : -1;
}

// L -> (t, r) with L = t * n_rho + r; n_rho is a power of two in every BASELINE config (rho_shift >= 0)
__device__ __forceinline__ void split_L(const DevParams& P, uint32_t L, int& t, int& r)
{
    if (P.rho_shift >= 0) { t = (int)(L >> P.rho_shift); r = (int)(L & ((1u << P.rho_shift) - 1u)); }
    else { t = (int)(L / (uint32_t)P.n_rho); r = (int)(L - (uint32_t)t * P.n_rho); }
}

__device__ __forceinline__ uint32_t hash_slot(uint32_t L, int nsbits) { return (L * 2654435761u) >> (32 - nsbits); }

__device__ __forceinline__ int hash_find(const uint32_t* keys, uint32_t L, int nsbits)
{
    const uint32_t msk = (1u << nsbits) - 1;
    uint32_t s = hash_slot(L, nsbits);
    while (true) {
        const uint32_t k = keys[s];
        if (k == L) return (int)s;
        if (k == kHashEmpty) return -1;
        s = (s + 1) & msk;
    }
}

// union-find over hash slots, 16-bit parents in shared memory (hook the larger root under the smaller one)
__device__ __forceinline__ uint32_t suf_find(volatile unsigned short* parent, uint32_t x)
{
    uint32_t p = parent[x];
    while (p != x) {
        const uint32_t gp = parent[p];
        if (gp == p) return p;
        parent[x] = (unsigned short)gp;  // path halving; x is not a root and never becomes one again
        x = gp;
        p = parent[x];
    }
    return x;
}

__device__ __forceinline__ void suf_union(unsigned short* parent, uint32_t a, uint32_t b)
{
    while (true) {
        a = suf_find(parent, a);
        b = suf_find(parent, b);
        if (a == b) return;
        if (a < b) { const uint32_t t = a; a = b; b = t; }
        const unsigned short old = atomicCAS(parent + a, (unsigned short)a, (unsigned short)b);
        if (old == (unsigned short)a) return;
    }
}

// ---------------------------------------------------------------- S1: voting (fast form)
//
// a' = u_q C + v_q S + O',  O' = O_q + (tile_base << sh),  sh = F - k,  row bytes = 2^k, tile_base a multiple of 2^k.
// For a hit that is in range at this theta, 0 <= a < n_rho 2^F, so as unsigned numbers
//     a' >> sh = (r << k) + (k fraction bits) + tile_base      with r = a >> F exactly,
// and masking the k low bits and OR-ing the lane's column offset gives the address of the counter word.

#define HOUGH_VOTE1(HX, HY)                                                                              \
    _Pragma("unroll") for (int g = 0; g < G; ++g) {                                                      \
        _Pragma("unroll") for (int j = 0; j < 2; ++j) {                                                  \
            const uint32_t a_ = (uint32_t)((HX) * C[g][j] + ((HY) * Sn[g][j] + Oq2));                    \
            red_add_shared(((a_ >> sh) & amask) | col[g], j ? 0x10000u : 1u);                            \
        }                                                                                                \
    }

template <int G>
__device__ __forceinline__ void fast_vote(const int2* __restrict__ hits, int n, int sh, uint32_t amask, int Oq2,
                                          const uint32_t (&col)[G], const int (&C)[G][2], const int (&Sn)[G][2])
{
    const int warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    const int4* h4 = reinterpret_cast<const int4*>(hits);
    const int npairs = n >> 1;
    int i = warp;
#pragma unroll 1
    for (; i + nwarps < npairs; i += 2 * nwarps) {  // four hits per trip: two 16-byte broadcast loads
        const int4 h0 = h4[i];
        const int4 h1 = h4[i + nwarps];
        HOUGH_VOTE1(h0.x, h0.y)
        HOUGH_VOTE1(h0.z, h0.w)
        HOUGH_VOTE1(h1.x, h1.y)
        HOUGH_VOTE1(h1.z, h1.w)
    }
    if (i < npairs) {
        const int4 h0 = h4[i];
        HOUGH_VOTE1(h0.x, h0.y)
        HOUGH_VOTE1(h0.z, h0.w)
    }
    if ((n & 1) && warp == nwarps - 1) {
        const int2 h = hits[n - 1];
        HOUGH_VOTE1(h.x, h.y)
    }
}
#undef HOUGH_VOTE1

// Checked form (hits that may leave the rho range at some theta, and strips that reach beyond n_theta).
template <int G>
__device__ __forceinline__ void checked_vote(const DevParams& P, const int2* __restrict__ hits, int first, int n, uint32_t tile_base,
                                             int k, const uint32_t (&col)[G], const int (&C)[G][2], const int (&Sn)[G][2],
                                             unsigned valid_bits)
{
    const int warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    const unsigned n_rho = (unsigned)P.n_rho;
    for (int i = first + warp; i < first + n; i += nwarps) {
        const int2 h = hits[i];
#pragma unroll
        for (int g = 0; g < G; ++g)
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                const int a = h.x * C[g][j] + (h.y * Sn[g][j] + P.Oq);
                const int r = a >> P.F;
                if ((unsigned)r < n_rho && ((valid_bits >> (2 * g + j)) & 1u))
                    red_add_shared(tile_base + ((uint32_t)r << k) + col[g], j ? 0x10000u : 1u);
            }
    }
}

// Count at (strip-local theta row tl, rho bin r) for the strip whose first theta row is `base`; rows -2 and -1 come from
// the halo saved from the previous strip; anything outside the grid counts as 0.
__device__ __forceinline__ uint32_t fcount_at(const DevParams& P, const uint16_t* tile, const uint16_t* halo, int base, int tl, int r)
{
    if ((unsigned)r >= (unsigned)P.n_rho) return 0;
    if (tl >= 0) return (tl < P.fS && base + tl < P.n_theta) ? tile[r * P.fS + tl] : 0;
    return halo[(tl + 2) * P.n_rho + r];
}

__device__ __forceinline__ bool fis_peak(const DevParams& P, const uint16_t* tile, const uint16_t* halo, int base, int tl, int r, uint32_t c)
{
    if (fcount_at(P, tile, halo, base, tl - 1, r - 1) >= c) return false;
    if (fcount_at(P, tile, halo, base, tl - 1, r) >= c) return false;
    if (fcount_at(P, tile, halo, base, tl - 1, r + 1) >= c) return false;
    if (fcount_at(P, tile, halo, base, tl, r - 1) >= c) return false;
    if (fcount_at(P, tile, halo, base, tl, r + 1) > c) return false;
    if (fcount_at(P, tile, halo, base, tl + 1, r - 1) > c) return false;
    if (fcount_at(P, tile, halo, base, tl + 1, r) > c) return false;
    if (fcount_at(P, tile, halo, base, tl + 1, r + 1) > c) return false;
    return true;
}

// ---------------------------------------------------------------- the fast event kernel

template <int G, int MAXT, int MINB>
__global__ void __launch_bounds__(MAXT, MINB)
hough_fast_kernel(const DevParams P, const float* __restrict__ u, const float* __restrict__ v,
                  const long long* __restrict__ offsets, int n_events, Candidate* __restrict__ cands, int* __restrict__ n_found)
{
    extern __shared__ __align__(1024) unsigned char smem[];
    // the control block sits at the end of the dynamic allocation: no static shared memory, so the tile starts the window
    FastShared& sh = *reinterpret_cast<FastShared*>(smem + P.f_off_kept + (size_t)P.K * 16);

    uint16_t* tile = reinterpret_cast<uint16_t*>(smem);
    int2* hits = reinterpret_cast<int2*>(smem + P.f_off_hits);
    uint16_t* halo = reinterpret_cast<uint16_t*>(smem + P.f_off_halo);
    uint32_t* slist = reinterpret_cast<uint32_t*>(smem + P.f_off_slist);  // strip list; later the tie list
    uint32_t* peaks = reinterpret_cast<uint32_t*>(smem + P.f_off_peaks);
    int* hist = reinterpret_cast<int*>(smem + P.f_off_hist);              // [256] peaks per min(votes, 255)
    uint32_t* kept = reinterpret_cast<uint32_t*>(smem + P.f_off_kept);    // [K] unordered, [K] sorted, [K] root slot, [K] size
    uint32_t* sorted = kept + P.K;
    uint32_t* kroot = sorted + P.K;
    uint32_t* ksize = kroot + P.K;
    // after the last strip the memory below f_off_kept is reused: hash keys [NS] u32, then parents [NS] u16
    uint32_t* hkeys = reinterpret_cast<uint32_t*>(smem);
    const int NS = 1 << P.fnsbits;
    unsigned short* hparent = reinterpret_cast<unsigned short*>(smem + (size_t)NS * 4);

    const int tid = threadIdx.x, nthr = blockDim.x, lane = tid & 31;
    const uint32_t tile_base = smem_addr(tile);
    const int k = P.fk, sh_amt = P.fsh, S = P.fS;
    const uint32_t amask = ~((1u << k) - 1u);
    const int Oq2 = P.Oq + (int)(tile_base << sh_amt);
    uint32_t col[G];
#pragma unroll
    for (int g = 0; g < G; ++g) col[g] = 4u * lane + 128u * g;
    const StageCtx sc{hits, &sh.n_safe, &sh.n_unsafe, P.fHB};
    uint32_t* onlist = P.f_onlist + (size_t)blockIdx.x * P.f_oncap;
    const uint32_t T = (uint32_t)P.T;
    const uint32_t TT = T | (T << 16);
    const int cpr = 8 * G;  // 16-byte chunks per rho row
#ifdef HOUGH_PHASE_TIMERS
    long long pt_acc[12] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
    long long pt_last = clock64();
#endif

    while (true) {
        __syncthreads();  // previous event fully done
        if (tid == 0) {
            sh.event = (int)atomicAdd(P.f_work_counter, 1u);
            sh.n_safe = 0; sh.n_unsafe = 0; sh.n_sl = 0; sh.n_on = 0; sh.n_peaks = 0; sh.n_kept = 0; sh.n_ties = 0; sh.defer = 0;
        }
        __syncthreads();
        const int e = sh.event;
        if (e >= n_events) break;

        const long long g0 = offsets[e], g1 = offsets[e + 1];
        const long long ne64 = g1 - g0;
        if (g0 < 0 || ne64 < 0 || ne64 > (long long)P.fHB || ne64 > (long long)P.max_hits_per_event) {
            // bad offsets, or more hits than the staging buffer: the general kernel handles (and flags) it
            if (tid == 0) P.deferred[atomicAdd(P.deferred_count, 1u)] = e;
            continue;
        }
        const int ne = (int)ne64;
        if (ne == 0) {  // an empty event has no on bins
            if (tid == 0) n_found[e] = 0;
            continue;
        }
        for (int i = tid; i < P.n_rho; i += nthr) reinterpret_cast<uint32_t*>(halo)[i] = 0;  // 2 rows of u16
        for (int i = tid; i < 256; i += nthr) hist[i] = 0;
        stage_hits(P, sc, u, v, g0, ne);
        HOUGH_PT(0);

        for (int strip = 0; strip < P.f_nstrips; ++strip) {
            const int base = strip * S;  // first theta row of the strip
            const bool last_strip = (strip == P.f_nstrips - 1);
            const bool full = base + S <= P.n_theta;
            {
                uint4* t4 = reinterpret_cast<uint4*>(tile);
                const int n16 = P.f_tile_bytes >> 4;
                for (int i = tid; i < n16; i += nthr) t4[i] = make_uint4(0, 0, 0, 0);
            }
            int C[G][2], Sn[G][2];
            unsigned valid_bits = 0;
#pragma unroll
            for (int g = 0; g < G; ++g)
#pragma unroll
                for (int j = 0; j < 2; ++j) {
                    const int tl = (g * 32 + lane) * 2 + j;
                    C[g][j] = __ldg(P.fCq + base + tl);
                    Sn[g][j] = __ldg(P.fSq + base + tl);
                    if (base + tl < P.n_theta) valid_bits |= 1u << (2 * g + j);
                }
            __syncthreads();  // tile zeroed, hits staged, strip list consumed
            HOUGH_PT(1);
            {
                const int ns = sh.n_safe, nu = sh.n_unsafe;
                if (full) fast_vote<G>(hits, ns, sh_amt, amask, Oq2, col, C, Sn);
                else checked_vote<G>(P, hits, 0, ns, tile_base, k, col, C, Sn, valid_bits);
                if (nu) checked_vote<G>(P, hits, P.fHB - nu, nu, tile_base, k, col, C, Sn, valid_bits);
            }
            __syncthreads();  // all votes of the strip are in
            HOUGH_PT(3);

            // ---------------- S2: threshold, compaction of the strip's on bins
            if (strip > 0) {  // deferred row: the last theta row of the previous strip, now that row 0 is known
                for (int r0 = tid - lane; r0 < P.n_rho; r0 += nthr) {
                    const int r = r0 + lane;
                    uint32_t c = 0;
                    bool pk = false;
                    if (r < P.n_rho) {
                        c = halo[P.n_rho + r];
                        pk = c >= T && fis_peak(P, tile, halo, base, -1, r, c);
                    }
                    const int i = warp_append(&sh.n_peaks, pk);
                    if (pk) {
                        if (i < P.fPCAP) peaks[i] = ((kCountMax - c) << kLBits) | (uint32_t)((base - 1) * P.n_rho + r);
                        atomicAdd(&hist[min(c, 255u)], 1);
                    }
                }
            }
            {
                const int total = P.n_rho * cpr;
                const uint4* t4 = reinterpret_cast<const uint4*>(tile);
                for (int i0 = tid - lane; i0 < total; i0 += nthr) {
                    const int idx = i0 + lane;
                    uint32_t m = 0;  // bit q set <=> count q of this chunk is on
                    uint4 w = make_uint4(0, 0, 0, 0);
                    if (idx < total) {
                        w = t4[idx];
                        const uint32_t gx = __vcmpgeu2(w.x, TT), gy = __vcmpgeu2(w.y, TT), gz = __vcmpgeu2(w.z, TT), gw = __vcmpgeu2(w.w, TT);
                        if (gx | gy | gz | gw) {
                            m = ((gx & 1u) | ((gx >> 15) & 2u)) | (((gy & 1u) | ((gy >> 15) & 2u)) << 2) |
                                (((gz & 1u) | ((gz >> 15) & 2u)) << 4) | (((gw & 1u) | ((gw >> 15) & 2u)) << 6);
                            if (!full) {  // theta rows beyond n_theta hold no votes, but keep the mask exact anyway
                                const int tl0 = (idx & (cpr - 1)) * 8;
                                for (int q = 0; q < 8; ++q) if (base + tl0 + q >= P.n_theta) m &= ~(1u << q);
                            }
                        }
                    }
                    if (__ballot_sync(0xffffffffu, m != 0) == 0) continue;
                    const int cnt = __popc(m);
                    int incl = cnt;
#pragma unroll
                    for (int o = 1; o < 32; o <<= 1) { const int y = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += y; }
                    int wbase = 0;
                    if (lane == 31) wbase = atomicAdd(&sh.n_sl, incl);
                    wbase = __shfl_sync(0xffffffffu, wbase, 31);
                    int slot = wbase + incl - cnt;
                    const int r = idx >> (k - 4), tl0 = (idx & (cpr - 1)) * 8;  // cpr = 2^(k-4) chunks per row
                    while (m) {
                        const int q = __ffs(m) - 1;
                        m &= m - 1;
                        const uint32_t wq = (q < 4) ? ((q < 2) ? w.x : w.y) : ((q < 6) ? w.z : w.w);
                        const uint32_t c = (wq >> (16 * (q & 1))) & 0xffffu;
                        if (c > kCountMax) sh.defer = 1;
                        // strip-list entry: bin index inside the tile (17 bits) | votes (10 bits)
                        if (slot < P.fSLCAP) slist[slot] = ((uint32_t)(r * S + tl0 + q) << kCountBits) | (c & kCountMax);
                        ++slot;
                    }
                }
            }
            __syncthreads();
            HOUGH_PT(4);
            // ---------------- one thread per on bin: global on list, local-maximum test
            {
                const int n_sl = sh.n_sl;
                const int on0 = sh.n_on;
                if (n_sl > P.fSLCAP) sh.defer = 1;  // benign race: every writer stores 1
                const int n_do = min(n_sl, P.fSLCAP);
                for (int i0 = tid - lane; i0 < n_do; i0 += nthr) {
                    const int i = i0 + lane;
                    bool pk = false;
                    uint32_t c = 0, L = 0;
                    if (i < n_do) {
                        const uint32_t ent = slist[i];
                        c = ent & kCountMax;
                        const int loc = (int)(ent >> kCountBits);
                        const int r = loc >> (k - 1), tl = loc & (S - 1);  // S = 2^(k-1) theta rows per strip
                        L = (uint32_t)((base + tl) * P.n_rho + r);
                        if (on0 + i < P.f_oncap) __stcg(onlist + on0 + i, L);
                        pk = (tl < S - 1 || last_strip) && fis_peak(P, tile, halo, base, tl, r, c);
                    }
                    const int ip = warp_append(&sh.n_peaks, pk);
                    if (pk) {
                        if (ip < P.fPCAP) peaks[ip] = ((kCountMax - c) << kLBits) | L;
                        atomicAdd(&hist[min(c, 255u)], 1);
                    }
                }
            }
            __syncthreads();
            HOUGH_PT(5);
            if (tid == 0) { sh.n_on += sh.n_sl; sh.n_sl = 0; }
            if (!last_strip) {  // keep the last two theta rows for the next strip's tests
                for (int r = tid; r < P.n_rho; r += nthr) {
                    halo[r] = tile[r * S + S - 2];
                    halo[P.n_rho + r] = tile[r * S + S - 1];
                }
            }
            __syncthreads();  // the tile may be zeroed again
            HOUGH_PT(6);
        }  // strips

        const int n_on = sh.n_on, n_pk = sh.n_peaks;
        if (sh.defer || n_on > P.f_oncap || n_pk > P.fPCAP) {
            if (tid == 0) P.deferred[atomicAdd(P.deferred_count, 1u)] = e;
            continue;
        }

        // ---------------- S4a: the K best peaks (key = (1023 - votes) << 22 | L, ascending)
        if (n_pk > P.K) {
            if (tid < 32) {  // threshold vote count c*: #(votes > c*) < K <= #(votes >= c*)
                int loc[8], s = 0;
#pragma unroll
                for (int j = 0; j < 8; ++j) { loc[j] = hist[255 - (lane * 8 + j)]; s += loc[j]; }  // descending votes
                int incl = s;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) { const int y = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += y; }
                int before = incl - s;
                if (before < P.K && P.K <= incl) {
                    int j = 0;
                    while (before + loc[j] < P.K) { before += loc[j]; ++j; }
                    sh.cstar = 255 - (lane * 8 + j);
                    sh.n_gt = before;
                }
            }
            __syncthreads();
            const int cstar = sh.cstar;
            if (cstar == 255) {  // bucket 255 lumps all larger counts together: not resolvable here
                if (tid == 0) P.deferred[atomicAdd(P.deferred_count, 1u)] = e;
                continue;
            }
            for (int i0 = tid - lane; i0 < n_pk; i0 += nthr) {
                const int i = i0 + lane;
                uint32_t key = 0;
                int c = -1;
                if (i < n_pk) { key = peaks[i]; c = (int)(kCountMax - (key >> kLBits)); }
                const int a = warp_append(&sh.n_kept, c > cstar);
                if (c > cstar) kept[a] = key;
                const int b = warp_append(&sh.n_ties, c == cstar);
                if (c == cstar && b < P.fSLCAP) slist[b] = key;
            }
            __syncthreads();
            const int n_ties = sh.n_ties, n_gt = sh.n_kept;
            if (n_ties > P.fSLCAP) {
                if (tid == 0) P.deferred[atomicAdd(P.deferred_count, 1u)] = e;
                continue;
            }
            const int need = P.K - n_gt;  // 1 <= need <= n_ties: the `need` smallest keys among the ties
            for (int i = tid; i < n_ties; i += nthr) {
                const uint32_t key = slist[i];
                int rank = 0;
                for (int j = 0; j < n_ties; ++j) rank += (slist[j] < key);
                if (rank < need) kept[n_gt + rank] = key;
            }
            if (tid == 0) sh.n_kept = P.K;
        } else {
            for (int i = tid; i < n_pk; i += nthr) kept[i] = peaks[i];
            if (tid == 0) sh.n_kept = n_pk;
        }
        __syncthreads();
        const int n_kept = sh.n_kept;
        for (int i = tid; i < n_kept; i += nthr) {  // slot = number of kept keys that are smaller (keys are unique)
            const uint32_t key = kept[i];
            int s = 0;
            for (int j = 0; j < n_kept; ++j) s += (kept[j] < key);
            sorted[s] = key;
            ksize[i] = 0;
        }
        __syncthreads();  // peaks, hist, strip list and tile are dead from here on
        HOUGH_PT(7);

        // ---------------- S3: connected components of the on mask: hash (L -> slot) + union-find over slots
        {
            uint4* h4 = reinterpret_cast<uint4*>(hkeys);
            for (int i = tid; i < NS / 4; i += nthr) h4[i] = make_uint4(kHashEmpty, kHashEmpty, kHashEmpty, kHashEmpty);
        }
        __syncthreads();
        const uint32_t hmsk = (uint32_t)NS - 1u;
        for (int i = tid; i < n_on; i += nthr) {
            const uint32_t L = __ldcg(onlist + i);
            uint32_t s = hash_slot(L, P.fnsbits);
            while (atomicCAS(hkeys + s, kHashEmpty, L) != kHashEmpty) s = (s + 1) & hmsk;
            hparent[s] = (unsigned short)s;
        }
        __syncthreads();
        HOUGH_PT(8);
        // NS and nthr are multiples of 32, so the trip count is warp-uniform; __syncwarp() makes the lanes reconverge after
        // the data-dependent probe / union loops of each trip (without it the warp stays split and runs lane by lane)
        for (int s = tid; s < NS; s += nthr) {
            const uint32_t L = hkeys[s];
            if (L != kHashEmpty) {
                int t, r;
                split_L(P, L, t, r);
                // the four neighbours with a smaller linear index; each adjacent pair is visited exactly once
                const uint32_t up = L - (uint32_t)P.n_rho;
                const int n0 = (r > 0) ? hash_find(hkeys, L - 1, P.fnsbits) : -1;
                const int n1 = (t > 0) ? hash_find(hkeys, up, P.fnsbits) : -1;
                const int n2 = (t > 0 && r > 0) ? hash_find(hkeys, up - 1, P.fnsbits) : -1;
                const int n3 = (t > 0 && r + 1 < P.n_rho) ? hash_find(hkeys, up + 1, P.fnsbits) : -1;
                if (n0 >= 0) suf_union(hparent, (uint32_t)s, (uint32_t)n0);
                if (n1 >= 0) suf_union(hparent, (uint32_t)s, (uint32_t)n1);
                else {  // (t-1, r-1) and (t-1, r+1) are already joined through (t-1, r) when that bin is on
                    if (n2 >= 0) suf_union(hparent, (uint32_t)s, (uint32_t)n2);
                    if (n3 >= 0) suf_union(hparent, (uint32_t)s, (uint32_t)n3);
                }
            }
            __syncwarp();
        }
        __syncthreads();
        HOUGH_PT(9);
        for (int s = tid; s < n_kept; s += nthr)
            kroot[s] = suf_find(hparent, (uint32_t)hash_find(hkeys, sorted[s] & kLMask, P.fnsbits));
        __syncthreads();
        for (int s = tid; s < n_kept; s += nthr) {
            const uint32_t root = kroot[s];
            int rs = 0;
            while (kroot[rs] != root) ++rs;  // best-ranked kept peak of the same component (<= s)
            // tag the root slot with rs + 1 in the 10 spare bits of its key (every peak of the component writes the same value)
            if (rs == s) hkeys[root] = (hkeys[root] & kLMask) | ((uint32_t)(rs + 1) << kLBits);
        }
        __syncthreads();
        for (int s = tid; s < NS; s += nthr) {  // sizes of the components that own a kept peak
            const uint32_t key = hkeys[s];
            if (key != kHashEmpty) {
                const uint32_t root = suf_find(hparent, (uint32_t)s);
                const uint32_t id = hkeys[root] >> kLBits;
                if (id != 0) atomicAdd(ksize + (id - 1), 1u);
            }
            __syncwarp();
        }
        __syncthreads();
        HOUGH_PT(10);

        // ---------------- S4b: records in rank order
        for (int s = tid; s < n_kept; s += nthr) {
            const uint32_t key = sorted[s];
            const uint32_t L = key & kLMask;
            const uint32_t c = kCountMax - (key >> kLBits);
            const uint32_t root = kroot[s];
            int rs = 0;
            while (kroot[rs] != root) ++rs;
            int t, r;
            split_L(P, L, t, r);
            const float th = (float)__ddiv_rn(__dmul_rn(3.14159265358979323846, (double)t), (double)P.n_theta);
            const float rho = (float)__dadd_rn(P.rho_min, __dmul_rn((double)r + 0.5, P.d_rho));
            int4* dst = reinterpret_cast<int4*>(cands + (size_t)e * P.K + s);
            dst[0] = make_int4(t, r, (int)c, rs);
            dst[1] = make_int4((int)ksize[rs], __float_as_int(th), __float_as_int(rho), 0);
        }
        if (tid == 0) n_found[e] = n_pk;
        HOUGH_PT(11);
    }
#ifdef HOUGH_PHASE_TIMERS
    if (threadIdx.x == 0)
        for (int q = 0; q < 12; ++q) atomicAdd(P.phase_cycles + q, (unsigned long long)pt_acc[q]);
#endif
}

}  // namespace hough
