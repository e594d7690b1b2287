// hough_fast.cuh -- the fast event kernel of libhough (sm_100a): vote + peaks + clusters with everything in shared memory.
//
// Same results as hough_event_kernel (hough_kernels.cuh), for the common case only; an event that does not fit the
// fast path's capacities is appended to a "deferred" list and processed afterwards by the general kernel:
//     more hits than the staged-hit buffer, a bin count above 1023, more on bins + on chunks in one strip than the
//     strip list holds, more on bins / peaks in the event than the parent / peak arrays hold, more ties at the K-th vote count
//     than the tie buffer.
//
// Per event (one CTA at a time):
//   S0  stage     fp32 hits -> fixed point, "safe" hits (in range for every theta) first             (O1)
//   per strip of S = 64 G theta rows (tile [n_rho][S] of u16 counters, theta fastest, row = 128 G bytes):
//   S1  vote      lane <-> 32-bit word column (2 theta rows), 2 IMAD + SHF + LOP3 + RED per vote:
//                 the tile base is folded into the fixed-point offset, so ((a >> (F - k)) & ~(2^k - 1)) | column
//                 IS the shared-memory address of the counter word                                   (Eq. 4.1)
//   S2  scan      pass 1 (sparse): 16-byte chunks (8 counts) -> list of the strip's on chunks, one ballot + one atomic per
//                 warp trip; the strip's last two theta rows are saved as the next strip's count halo on the way
//                 pass 2 (dense): one thread per on chunk: (a) strict-local-maximum test of its 8 bins at once on packed
//                 halfwords, straight from the counts (1 theta row of halo kept between strips)        (L94, L106)
//                 -> per-bin strip-list entries (peak flag | offset to the run's head | tile index | votes)
//                 (b) the on bin's tile entry is overwritten with 0x8000 | its index in the event's on list
//   S3  clusters  (c) each on bin reads the entries of its four earlier neighbours straight from the tile and joins
//                 them in a union-find over on-list indices (16-bit parents in shared memory)         (keyword L29)
//   then, once per event:
//   S4  select    vote-count histogram -> threshold count -> ties ranked by index -> K best peaks; component sizes
//                 of the kept peaks' components; 32-byte records in rank order
#pragma once
#include "hough_kernels.cuh"

namespace hough {

constexpr uint32_t kOnFlag = 0x8000u;  // tile entry of an on bin after step (b): kOnFlag | on-list index
constexpr int kCountBits = 10;  // packed peak key: (1023 - votes) << 22 | L   (smaller key = better rank)
constexpr uint32_t kCountMax = (1u << kCountBits) - 1;

struct FastShared {  // static shared control block
    int event;
    int n_safe, n_unsafe;
    int n_ch;     // on chunks of the current strip (grow down from the end of the strip list)
    int n_sl;     // on bins of the current strip (strip list)
    int n_on;     // on bins of the event so far (global on list)
    int n_peaks;  // peaks of the event so far
    int n_kept, n_ties;
    int n_final;  // records of the event after selection (n_kept is still being read when this is written)
    int defer;
    int cstar, n_gt;  // threshold vote count and number of peaks above it
    unsigned int r2max;  // max over the event's valid hits of u_q^2 + v_q^2
};

__device__ __forceinline__ unsigned lanemask_lt()
{
#ifdef HOUGH_EMU
    return (1u << (threadIdx.x & 31)) - 1u;
#else
    unsigned m;
    asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
    return m;
#endif
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

// union-find over on-list indices, 16-bit parents in shared memory (hook the larger root under the smaller one)
__device__ __forceinline__ uint32_t suf_find(const DevParams& P, volatile unsigned short* parent, uint32_t x)
{
    if (!HB(P, x, P.f_oncap, 110)) return 0;
    uint32_t p = parent[x];
    while (p != x) {
        if (!HB(P, p, P.f_oncap, 111)) return 0;
        const uint32_t gp = parent[p];
        if (!HB(P, gp, P.f_oncap, 112)) return 0;
        if (gp == p) return p;
        parent[x] = (unsigned short)gp;  // path halving; x is not a root and never becomes one again
        x = gp;
        p = parent[x];
    }
    return x;
}

__device__ __forceinline__ void suf_union(const DevParams& P, unsigned short* parent, uint32_t a, uint32_t b)
{
    while (true) {
        a = suf_find(P, parent, a);
        b = suf_find(P, parent, b);
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
            const uint32_t ad_ = ((a_ >> sh) & amask) | col[g];                                          \
            if (HB(P, ad_ - vt_base, vt_bytes, 101)) red_add_shared(ad_, j ? 0x10000u : 1u);             \
        }                                                                                                \
    }

template <int G, int NW>
__device__ __forceinline__ void fast_vote(const DevParams& P, uint32_t vt_base, const int2* __restrict__ hits, int n, int sh, uint32_t amask, int Oq2,
                                          const uint32_t (&col)[G], const int (&C)[G][2], const int (&Sn)[G][2])
{
    const uint32_t vt_bytes = (uint32_t)P.f_tile_bytes;  // used by the -DHOUGH_BOUNDS build only
    (void)vt_base; (void)vt_bytes;
    // Hits are sliced over the NW warps of the CTA two at a time (one 16-byte broadcast load); a trip takes four such
    // pairs (the loads carry their strides as immediates), so the loop overhead is 7 instructions per 32 G votes.
    const int warp = threadIdx.x >> 5;
    const int npairs = n >> 1;
    if ((n & 1) && warp == NW - 1) {  // odd last hit
        const int2 h = hits[n - 1];
        HOUGH_VOTE1(h.x, h.y)
    }
    const int4* p = reinterpret_cast<const int4*>(hits) + warp;
    int i = warp;
#pragma unroll 1
    for (; i + 7 * NW < npairs; i += 8 * NW, p += 8 * NW) {
#pragma unroll
        for (int hh = 0; hh < 2; ++hh) {
            const int4 h0 = p[(4 * hh) * NW], h1 = p[(4 * hh + 1) * NW], h2 = p[(4 * hh + 2) * NW], h3 = p[(4 * hh + 3) * NW];
            HOUGH_VOTE1(h0.x, h0.y)
            HOUGH_VOTE1(h0.z, h0.w)
            HOUGH_VOTE1(h1.x, h1.y)
            HOUGH_VOTE1(h1.z, h1.w)
            HOUGH_VOTE1(h2.x, h2.y)
            HOUGH_VOTE1(h2.z, h2.w)
            HOUGH_VOTE1(h3.x, h3.y)
            HOUGH_VOTE1(h3.z, h3.w)
        }
    }
#pragma unroll 1
    for (; i < npairs; i += NW, p += NW) {
        const int4 h0 = p[0];
        HOUGH_VOTE1(h0.x, h0.y)
        HOUGH_VOTE1(h0.z, h0.w)
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
                if ((unsigned)r < n_rho && ((valid_bits >> (2 * g + j)) & 1u) && HB(P, ((uint32_t)r << k) + col[g], P.f_tile_bytes, 102))
                    red_add_shared(tile_base + ((uint32_t)r << k) + col[g], j ? 0x10000u : 1u);
            }
    }
}

// Tile entry of bin (strip-local theta row tl, rho bin r) after step (b): kOnFlag | on-list index for an on bin, a
// count below the threshold otherwise.  Row -1 is the previous strip's last row (index halo); outside the grid -> 0.
__device__ __forceinline__ uint32_t fentry_at(const DevParams& P, const uint16_t* tile, const uint16_t* ihalo_prev, int tl, int r)
{
    if ((unsigned)r >= (unsigned)P.n_rho) return 0;
    return tl >= 0 ? tile[r * P.fS + tl] : ihalo_prev[r];
}

// ---------------------------------------------------------------- the fast event kernel

// One vote-count histogram update per distinct count in the warp (peaks of an event share a handful of counts, and
// same-address shared-memory atomics serialise).  Every lane of the warp must call.
__device__ __forceinline__ void hist_add(int* hist, bool pk, uint32_t c)
{
    const unsigned pm = __ballot_sync(0xffffffffu, pk);
    if (pk) {
        const uint32_t cb = min(c, 255u);
        const unsigned same = __match_any_sync(pm, cb);
        if ((int)(threadIdx.x & 31) == __ffs(same) - 1) atomicAdd(&hist[cb], __popc(same));
    }
}

template <int G, int MAXT, int MINB>
__global__ void __launch_bounds__(MAXT, MINB)
hough_fast_kernel(const DevParams P, const float* __restrict__ u, const float* __restrict__ v,
                  const long long* __restrict__ offsets, int n_events, Candidate* __restrict__ cands, int* __restrict__ n_found)
{
    HOUGH_DYNAMIC_SMEM(smem);
    // the control block sits at the end of the dynamic allocation: no static shared memory, so the tile starts the window
    FastShared& sh = *reinterpret_cast<FastShared*>(smem + P.f_off_kept + (size_t)P.K * 20);

    uint16_t* tile = reinterpret_cast<uint16_t*>(smem);
    int2* hits = reinterpret_cast<int2*>(smem + P.f_off_hits);
    uint16_t* halo = reinterpret_cast<uint16_t*>(smem + P.f_off_halo);      // [2][2][n_rho] counts of a strip's last two rows, by strip parity
    uint16_t* ihalo = reinterpret_cast<uint16_t*>(smem + P.f_off_ihalo);    // [2][n_rho] entries of a strip's last row, by strip parity
    uint32_t* slist = reinterpret_cast<uint32_t*>(smem + P.f_off_slist);    // strip list; later the tie list
    uint32_t* peaks = reinterpret_cast<uint32_t*>(smem + P.f_off_peaks);    // [PCAP] packed keys
    uint16_t* pidx = reinterpret_cast<uint16_t*>(smem + P.f_off_pidx);      // [PCAP] on-list index of each peak
    unsigned short* parent = reinterpret_cast<unsigned short*>(smem + P.f_off_parent);  // [ONCAP]
    int* hist = reinterpret_cast<int*>(smem + P.f_off_hist);                // [256] peaks per min(votes, 255)
    uint32_t* kept = reinterpret_cast<uint32_t*>(smem + P.f_off_kept);      // [K] each: unordered keys, sorted keys, roots, sizes
    uint32_t* sorted = kept + P.K;
    uint32_t* kroot = sorted + P.K;
    uint32_t* ksize = kroot + P.K;
    uint16_t* kidx = reinterpret_cast<uint16_t*>(ksize + P.K);              // [K] on-list index, unordered / sorted
    uint16_t* sidx = kidx + P.K;
    uint32_t* roottag = reinterpret_cast<uint32_t*>(tile);  // after the last strip: [ONCAP] K - slot of the best kept peak, at roots

    const int tid = threadIdx.x, nthr = blockDim.x, lane = tid & 31;
    const uint32_t tile_base = smem_addr(tile);
    const int k = P.fk, sh_amt = P.fsh, S = P.fS;
    uint32_t amask = ~((1u << k) - 1u);
    int sh_reg = sh_amt;
    asm volatile("" : "+r"(amask), "+r"(sh_reg));  // per-thread registers (not uniform-datapath operands) for the vote loop
    const int Oq2 = P.Oq + (int)(tile_base << sh_amt);
    uint32_t col[G];
    // 128 bytes between a lane's word columns, taken from a kernel parameter (2 fS / G with fS = 64 G): ptxas cannot
    // fold col[g] back into col[0] | constant, so ((a >> sh) & mask) | col[g] stays ONE LOP3 per vote for every g
    const uint32_t col_stride = (uint32_t)(2 * P.fS) / (uint32_t)G;
#pragma unroll
    for (int g = 0; g < G; ++g) col[g] = 4u * lane + col_stride * g;
    const StageCtx sc{hits, &sh.n_safe, &sh.n_unsafe, P.fHB, &sh.r2max};
    const uint32_t T = (uint32_t)P.T;
    const uint32_t tadd = (0x8000u - T) * 0x00010001u;
    const uint32_t oadd = (0x8000u - (kCountMax + 1u)) * 0x00010001u;
    const int cpr = 8 * G;  // 16-byte chunks per rho row
#ifdef HOUGH_PHASE_TIMERS
    long long pt_acc[12] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
    long long pt_last = clock64();
#endif

    // The address folding of the vote (Oq2) is valid only if the tile starts below 4096 in the shared window and on a row
    // boundary (the host sized the fixed-point range for that).  If the driver ever places it elsewhere, nothing is
    // computed here: every event this CTA fetches goes to the general kernel.
    const bool fold_ok = tile_base < 4096u && (tile_base & ((1u << k) - 1u)) == 0u;
    // Dense workloads (every bin on: e.g. 2000 hits on a 128 x 128 grid) overflow the lists event after event; the vote spent on
    // such an event is wasted, the general kernel redoes it.  After kGiveUpRun capacity overflows in a row this CTA hands the next
    // kGiveUpSkip events over untouched, then tries again.  Block-uniform registers; changes which kernel computes an event, never a result.
    constexpr int kGiveUpRun = 8, kGiveUpSkip = 64;
    int overflow_run = 0, skip_left = 0;

    while (true) {
        __syncthreads();  // previous event fully done
        if (tid == 0) {
            sh.event = (int)atomicAdd(P.f_work_counter, 1u);
            sh.n_safe = 0; sh.n_unsafe = 0; sh.n_ch = 0; sh.n_sl = 0; sh.n_on = 0; sh.n_peaks = 0; sh.n_kept = 0; sh.n_ties = 0; sh.defer = 0;
        }
        __syncthreads();
        const int e = sh.event;
        if (e >= n_events) break;

        const long long g0 = offsets[e], g1 = offsets[e + 1];
        const long long ne64 = g1 - g0;
        if (skip_left > 0 && ne64 > 0) {
            --skip_left;
            if (tid == 0) P.deferred[atomicAdd(P.deferred_count, 1u)] = e;
            continue;
        }
        if (!fold_ok || g0 < 0 || ne64 < 0 || g1 > P.max_hits || ne64 > (long long)P.fHB || ne64 > (long long)P.max_hits_per_event) {
            // bad offsets, or more hits than the staging buffer: the general kernel handles (and flags) it
            if (tid == 0) P.deferred[atomicAdd(P.deferred_count, 1u)] = e;
            continue;
        }
        const int ne = (int)ne64;
        if (ne == 0) {  // an empty event has no on bins
            if (tid == 0) n_found[e] = 0;
            continue;
        }
        for (int i = tid; i < P.n_rho; i += nthr) {  // count halos (2 x 2 rows) and index halos (2 rows), as u16 pairs
            reinterpret_cast<uint32_t*>(halo)[i] = 0;
            reinterpret_cast<uint32_t*>(halo)[P.n_rho + i] = 0;
            reinterpret_cast<uint32_t*>(ihalo)[i] = 0;
        }
        if (tid == 0) sh.r2max = 0u;
        for (int i = tid; i < 256; i += nthr) hist[i] = 0;
        __syncthreads();
        stage_hits(P, sc, u, v, g0, ne);
        HOUGH_PT(0);
        int r_lo = 0, r_hi = P.n_rho - 1;  // rho rows some vote of this event can reach (set after the first strip's barrier)

        bool give_up = false;
        for (int strip = 0; strip < P.f_nstrips; ++strip) {
            const int base = strip * S;  // first theta row of the strip
            const bool last_strip = (strip == P.f_nstrips - 1);
            const bool full = base + S <= P.n_theta;
            const uint16_t* ihalo_prev = ihalo + ((strip + 1) & 1) * P.n_rho;  // written by the previous strip
            uint16_t* ihalo_cur = ihalo + (strip & 1) * P.n_rho;
            const uint16_t* halo_prev = halo + ((strip + 1) & 1) * 2 * P.n_rho;
            uint16_t* halo_cur = halo + (strip & 1) * 2 * P.n_rho;
            {   // strip 0 clears the whole tile (rows outside [r_lo, r_hi] then stay clear for the event), later strips the
                // reachable rows plus one on each side (the neighbourhood tests read them)
                uint4* t4 = reinterpret_cast<uint4*>(tile);
                const int z_lo = strip == 0 ? 0 : max(r_lo - 1, 0) * cpr, z_hi = strip == 0 ? (P.f_tile_bytes >> 4) : min(r_hi + 2, P.n_rho) * cpr;
                for (int i = z_lo + tid; i < z_hi; i += nthr) t4[i] = make_uint4(0, 0, 0, 0);
                for (int i = tid; i < P.n_rho; i += nthr) ihalo_cur[i] = 0;  // filled by step (b)
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
            __syncthreads();  // tile zeroed, hits staged
            if (strip == 0) {
                // |u_q C + v_q S| <= (M + 1) sqrt(u_q^2 + v_q^2) for every theta (Cauchy-Schwarz; the table entries are within 1/2 of
                // M cos, M sin), so all votes of the event fall into rows [(O_q - B) >> F, (O_q + B) >> F]
                // (stage_one clamps r2max at 2^32 - 1: a clamped value bounds nothing, every row stays reachable)
                if (sh.r2max != 0xffffffffu) {
                    const long long B = (long long)P.Mq1 * ((long long)ceil(sqrt((double)sh.r2max)) + 1);
                    r_lo = (int)max(((long long)P.Oq - B) >> P.F, 0ll);
                    r_hi = (int)min(((long long)P.Oq + B) >> P.F, (long long)P.n_rho - 1);
                    if (r_lo > r_hi) { r_lo = 0; r_hi = P.n_rho - 1; }
                }
            }
            HOUGH_PT(1);
            {
                const int ns = sh.n_safe, nu = sh.n_unsafe;
                if (full) fast_vote<G, MAXT / 32>(P, tile_base, hits, ns, sh_reg, amask, Oq2, col, C, Sn);  // launched with MAXT threads
                else checked_vote<G>(P, hits, 0, ns, tile_base, k, col, C, Sn, valid_bits);
                if (nu) checked_vote<G>(P, hits, P.fHB - nu, nu, tile_base, k, col, C, Sn, valid_bits);
            }
            __syncthreads();  // all votes of the strip are in
            HOUGH_PT(3);

            // ---------------- S2: threshold.  Pass 1 (sparse: one warp trip in two finds nothing) only appends the on CHUNKS
            // (chunk index | on mask << 16) to a list that grows down from the end of the strip list: one ballot, one atomic
            // per warp trip.  Pass 2 (dense: one thread per on chunk) expands them into the strip list's per-bin entries.
            {
                // nthr is a multiple of cpr, so a thread stays in one chunk column: its shared-memory address and its halo slot
                // advance by constants, and only the threads of the last chunk column save the count halo
                const int i_lo = r_lo * cpr, i_hi = (r_hi + 1) * cpr;  // only rho rows some hit can reach
                const bool halo_lane = (tid & (cpr - 1)) == cpr - 1;
                uint16_t* hp = halo_cur + r_lo + tid / cpr;
                const uint32_t a_end = tile_base + 16u * (uint32_t)i_hi;
                for (uint32_t a = tile_base + 16u * (uint32_t)(i_lo + tid); a - 16u * lane < a_end; a += 16u * nthr, hp += nthr / cpr) {
                    uint32_t m = 0;  // bit q set <=> count q of this chunk is on
                    if (a < a_end && HB(P, a - tile_base, P.f_tile_bytes, 122)) {
                        const uint4 w = lds128(a);
                        // counts are below 2^15 (at most one vote per hit, fHB <= 32767), so adding 2^15 - T to both
                        // halfwords sets their top bits exactly where count >= T, without a carry between them
                        const uint32_t gx = (w.x + tadd) & 0x80008000u, gy = (w.y + tadd) & 0x80008000u;
                        const uint32_t gz = (w.z + tadd) & 0x80008000u, gw = (w.w + tadd) & 0x80008000u;
                        if (gx | gy | gz | gw) {
                            m = (((gx >> 15) | (gx >> 30)) & 3u) | ((((gy >> 15) | (gy >> 30)) & 3u) << 2) |
                                ((((gz >> 15) | (gz >> 30)) & 3u) << 4) | ((((gw >> 15) | (gw >> 30)) & 3u) << 6);
                            // a count above 1023 does not fit the packed entries: the general kernel takes the event
                            if (((w.x + oadd) | (w.y + oadd) | (w.z + oadd) | (w.w + oadd)) & 0x80008000u) atomicOr(&sh.defer, 1);  // several threads may: no plain store
                        }
                        // theta rows beyond n_theta hold no votes (checked_vote masks them), so m needs no masking
                        if (halo_lane && HB(P, hp - halo_cur, P.n_rho, 120)) {  // the row's two last counts are the next strip's count halo
                            hp[0] = (uint16_t)(w.w & 0xffffu);  // (rows no vote can reach are never scanned: they stay 0 from the event's start)
                            hp[P.n_rho] = (uint16_t)(w.w >> 16);
                        }
                    }
                    const unsigned bal = __ballot_sync(0xffffffffu, m != 0);
                    if (bal == 0) continue;
                    int cb = 0;
                    if (lane == 0) cb = atomicAdd(&sh.n_ch, __popc(bal));
                    cb = __shfl_sync(0xffffffffu, cb, 0) + __popc(bal & lanemask_lt());
                    if (m != 0 && cb < P.fSLCAP && HB(P, P.fSLCAP - 1 - cb, P.fSLCAP, 121)) slist[P.fSLCAP - 1 - cb] = ((a - tile_base) >> 4) | (m << 16);
                }
            }
            __syncthreads();
            const int n_ch = sh.n_ch;
            if (sh.defer || n_ch > P.fSLCAP) { give_up = true; break; }  // block-uniform
            const int sl_lim = P.fSLCAP - n_ch;  // per-bin entries fill [0, sl_lim), the chunk list sits behind them
            // One thread per on chunk (8 consecutive theta rows of one rho row).  The counts are still intact, so the strict
            // local-maximum test (O4) is done here for the 8 bins at once on packed halfwords: with a / b / c the counts of rho
            // rows r-1 / r / r+1 and V[q] = max(a[q], b[q], c[q]),
            //     peak(q) <=> on(q) and b[q] > max(V[q-1], a[q]) and b[q] >= max(V[q+1], c[q])
            // (the neighbours of smaller linear index must be beaten, the others matched).  A bin of the strip's last theta
            // row waits for the next strip ("deferred row" below) unless this is the last strip.
            for (int j0 = tid - lane; j0 < n_ch; j0 += nthr) {
                const int j = j0 + lane;
                uint32_t m = 0, loc0 = 0, pk8 = 0;
                uint4 Bw = make_uint4(0, 0, 0, 0);
                if (j < n_ch && HB(P, (slist[P.fSLCAP - 1 - j] & 0xffffu), P.f_tile_bytes >> 4, 123)) {
                    const uint32_t ce = slist[P.fSLCAP - 1 - j];
                    m = ce >> 16;
                    const int cidx = (int)(ce & 0xffffu);
                    loc0 = (uint32_t)cidx << 3;  // chunk idx holds the tile halfwords 8 idx ... 8 idx + 7
                    const int r = cidx / cpr, cq = cidx & (cpr - 1);
                    const bool up = r > 0, dn = r + 1 < P.n_rho;
                    const uint4* t4 = reinterpret_cast<const uint4*>(tile);
                    const uint4 z4 = make_uint4(0, 0, 0, 0);
                    Bw = t4[cidx];
                    const uint4 Aw = up ? t4[cidx - cpr] : z4, Cw = dn ? t4[cidx + cpr] : z4;
                    uint32_t em, ep = 0;  // max of the three counts one theta row before / after the chunk
                    if (cq > 0) {
                        const uint16_t* e = tile + loc0 - 1;
                        em = max((uint32_t)e[0], max(up ? (uint32_t)e[-S] : 0u, dn ? (uint32_t)e[S] : 0u));
                    } else {  // the previous strip's last theta row (all zero for the first strip)
                        const uint16_t* e = halo_prev + P.n_rho + r;
                        em = max((uint32_t)e[0], max(up ? (uint32_t)e[-1] : 0u, dn ? (uint32_t)e[1] : 0u));
                    }
                    if (cq < cpr - 1) {
                        const uint16_t* e = tile + loc0 + 8;
                        ep = max((uint32_t)e[0], max(up ? (uint32_t)e[-S] : 0u, dn ? (uint32_t)e[S] : 0u));
                    }
                    const uint32_t V0 = __vmaxu2(__vmaxu2(Aw.x, Bw.x), Cw.x), V1 = __vmaxu2(__vmaxu2(Aw.y, Bw.y), Cw.y);
                    const uint32_t V2 = __vmaxu2(__vmaxu2(Aw.z, Bw.z), Cw.z), V3 = __vmaxu2(__vmaxu2(Aw.w, Bw.w), Cw.w);
                    // Vm_j = (V[2j-1], V[2j]): the column maxima one theta row up; one theta row down it is Vm_(j+1)
                    const uint32_t Vm0 = __byte_perm(em << 16, V0, 0x5432), Vm1 = __byte_perm(V0, V1, 0x5432);
                    const uint32_t Vm2 = __byte_perm(V1, V2, 0x5432), Vm3 = __byte_perm(V2, V3, 0x5432), Vm4 = __byte_perm(V3, ep, 0x5432);
                    // counts are below 2^15: (b | 2^15) - x keeps bit 15 exactly where b >= x, without a borrow between the halfwords
                    auto pkw = [](uint32_t bw, uint32_t sm, uint32_t nm) -> uint32_t {
                        const uint32_t bh = bw | 0x80008000u;
                        return (bh - sm - 0x00010001u) & (bh - nm) & 0x80008000u;
                    };
                    const uint32_t gx = pkw(Bw.x, __vmaxu2(Vm0, Aw.x), __vmaxu2(Vm1, Cw.x)), gy = pkw(Bw.y, __vmaxu2(Vm1, Aw.y), __vmaxu2(Vm2, Cw.y));
                    const uint32_t gz = pkw(Bw.z, __vmaxu2(Vm2, Aw.z), __vmaxu2(Vm3, Cw.z)), gw = pkw(Bw.w, __vmaxu2(Vm3, Aw.w), __vmaxu2(Vm4, Cw.w));
                    pk8 = (((gx >> 15) | (gx >> 30)) & 3u) | ((((gy >> 15) | (gy >> 30)) & 3u) << 2) |
                          ((((gz >> 15) | (gz >> 30)) & 3u) << 4) | ((((gw >> 15) | (gw >> 30)) & 3u) << 6);
                    pk8 &= m;
                    if (cq == cpr - 1 && !last_strip) pk8 &= 0x7fu;  // its lower neighbours are in the next strip
                }
                const int cnt = __popc(m);
                int incl = cnt;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) { const int y = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += y; }
                int wbase = 0;
                if (lane == 31) wbase = atomicAdd(&sh.n_sl, incl);
                wbase = __shfl_sync(0xffffffffu, wbase, 31);
                int slot = wbase + incl - cnt;
                uint32_t head = 0;  // offset back to the first bin of the run of on bins (consecutive theta rows) that contains q
                uint32_t prev = 0xfffffff0u;  // prev + 1 matches no bit position
                while (m) {
                    const int q = __ffs(m) - 1;
                    m &= m - 1;
                    head = ((uint32_t)q == prev + 1u) ? head + 1u : 0u;
                    prev = (uint32_t)q;
                    const uint32_t c = (uint32_t)tile[loc0 + q] & kCountMax;
                    // strip-list entry: peak (bit 30) | offset back to its run's head (3 bits) | bin index inside the tile (17 bits) | votes (10 bits)
                    if (slot < sl_lim && HB(P, slot, P.fSLCAP, 124)) slist[slot] = (((pk8 >> q) & 1u) << 30) | (head << 27) | ((loc0 + q) << kCountBits) | c;
                    ++slot;
                }
            }
            __syncthreads();
            HOUGH_PT(4);
            const int n_sl = sh.n_sl, on0 = sh.n_on;
            if (n_sl > sl_lim || on0 + n_sl > P.f_oncap) { give_up = true; break; }  // block-uniform

            // ---------------- (b) on bins become kOnFlag | on-list index; a bin below another on bin of its chunk joins that
            //                      run's head right away (indices of one chunk are consecutive), the others are singletons
            for (int i = tid; i < n_sl; i += nthr) {
                const uint32_t ent = slist[i];
                const uint32_t loc = (ent >> kCountBits) & 0x1ffffu;
                const uint16_t en = (uint16_t)(kOnFlag | (uint32_t)(on0 + i));
                if (!HB(P, loc, P.f_tile_bytes >> 1, 130) || !HB(P, on0 + i, P.f_oncap, 131)) continue;
                tile[loc] = en;
                if ((loc & (uint32_t)(S - 1)) == (uint32_t)(S - 1) && HB(P, loc >> (k - 1), P.n_rho, 132)) ihalo_cur[loc >> (k - 1)] = en;  // last theta row: index halo of the next strip
                parent[on0 + i] = (unsigned short)(on0 + i - (int)((ent >> 27) & 7u));  // the head of its run inside the chunk
            }
            __syncthreads();
            HOUGH_PT(5);

            // ---------------- (c) one thread per on bin: S3 joins from the entries of its four neighbours of smaller linear index;
            // the peak flag comes with the strip-list entry.  A neighbour's count, where the deferred row needs it, is in the
            // strip list (this strip) or in the count halo (previous strip's last row).
            auto ncount = [&](uint32_t en, int tl_nb, int r_nb) -> uint32_t {
                if (!(en & kOnFlag)) return 0u;
                if (tl_nb >= 0 && !HB(P, (int)(en & 0x7fffu) - on0, n_sl, 140)) return 0u;
                return tl_nb >= 0 ? (slist[(int)(en & 0x7fffu) - on0] & kCountMax) : (uint32_t)halo_prev[P.n_rho + r_nb];
            };
            // Lane l of a warp takes entry l * W + (warp-trip index): the 32 lanes of a warp work on 32 far-apart bins and do
            // not fight over one root.  The trips start at the last warp: the first ones have the deferred row to do.
            const int W = (n_sl + 31) >> 5;
            for (int i0 = nthr - 32 - (tid - lane); i0 < W * 32; i0 += nthr) {
                const int i = lane * W + (i0 >> 5);
                bool pk = false;
                uint32_t c = 0, L = 0, q0 = 0xffffffffu, q1 = 0xffffffffu, me_idx = 0;
                if (i < n_sl) {
                    const uint32_t ent = slist[i];
                    c = ent & kCountMax;
                    pk = (ent >> 30) & 1u;
                    const int loc = (int)((ent >> kCountBits) & 0x1ffffu), hoff = (int)((ent >> 27) & 7u);
                    const int r = loc >> (k - 1), tl = loc & (S - 1);  // S = 2^(k-1) theta rows per strip
                    const uint32_t me = (uint32_t)(on0 + i);
                    L = (uint32_t)((base + tl) * P.n_rho + r);
                    const uint32_t n0 = fentry_at(P, tile, ihalo_prev, tl, r - 1);
                    const uint32_t n1 = hoff > 0 ? kOnFlag : fentry_at(P, tile, ihalo_prev, tl - 1, r);
                    const uint32_t n2 = fentry_at(P, tile, ihalo_prev, tl - 1, r - 1);
                    const uint32_t n3 = fentry_at(P, tile, ihalo_prev, tl - 1, r + 1);
                    // a join is skipped when other joins already imply it.  At most two partners remain; they go through ONE
                    // union call site so that the lanes of a warp stay together.
                    constexpr uint32_t kNone = 0xffffffffu;
                    if (n1 & kOnFlag) {
                        if (hoff == 0) q0 = n1 & 0x7fffu;
                        if ((n0 & kOnFlag) && !(n2 & kOnFlag)) q1 = n0 & 0x7fffu;
                    } else {
                        if (n0 & kOnFlag) q0 = n0 & 0x7fffu;
                        else if (n2 & kOnFlag) q0 = n2 & 0x7fffu;
                        if (n3 & kOnFlag) q1 = n3 & 0x7fffu;
                    }
                    if (q0 == kNone) { q0 = q1; q1 = kNone; }
                    me_idx = me;
                }
#pragma unroll 1
                for (int kk = 0; kk < 2; ++kk) {
                    const uint32_t q = kk ? q1 : q0;
                    if (q != 0xffffffffu && HB(P, q, on0 + n_sl, 141)) suf_union(P, parent, me_idx, q);
                    if (__ballot_sync(0xffffffffu, q1 != 0xffffffffu) == 0) break;  // warp-uniform
                }
                __syncwarp();  // reconverge after the data-dependent union loops
                const int ip = warp_append(&sh.n_peaks, pk);
                if (pk) {
                    if (ip < P.fPCAP && HB(P, ip, P.fPCAP, 142)) { peaks[ip] = ((kCountMax - c) << kLBits) | L; pidx[ip] = (uint16_t)(on0 + i); }
                }
                hist_add(hist, pk, c);
            }
            HOUGH_PT(2);
            if (strip > 0) {  // deferred row: the last theta row of the previous strip, now that row 0 of this one is known
                for (int r0 = tid - lane; r0 < P.n_rho; r0 += nthr) {
                    const int r = r0 + lane;
                    uint32_t c = 0;
                    bool pk = false;
                    if (r < P.n_rho) {
                        c = halo_prev[P.n_rho + r];
                        if (c >= T) {
                            const uint32_t lft = r > 0 ? halo_prev[P.n_rho + r - 1] : 0u, rgt = r + 1 < P.n_rho ? halo_prev[P.n_rho + r + 1] : 0u;
                            const uint32_t a0 = r > 0 ? halo_prev[r - 1] : 0u, a1 = halo_prev[r], a2 = r + 1 < P.n_rho ? halo_prev[r + 1] : 0u;
                            pk = a0 < c && a1 < c && a2 < c && lft < c && rgt <= c &&
                                 ncount(fentry_at(P, tile, ihalo_prev, 0, r - 1), 0, r - 1) <= c &&
                                 ncount(fentry_at(P, tile, ihalo_prev, 0, r), 0, r) <= c &&
                                 ncount(fentry_at(P, tile, ihalo_prev, 0, r + 1), 0, r + 1) <= c;
                        }
                    }
                    const int ip = warp_append(&sh.n_peaks, pk);
                    if (pk) {
                        if (ip < P.fPCAP && HB(P, ip, P.fPCAP, 143)) {
                            peaks[ip] = ((kCountMax - c) << kLBits) | (uint32_t)((base - 1) * P.n_rho + r);
                            pidx[ip] = (uint16_t)(ihalo_prev[r] & 0x7fffu);
                        }
                    }
                    hist_add(hist, pk, c);
                }
            }
            HOUGH_PT(9);
            if (tid == 0) { sh.n_on = on0 + n_sl; sh.n_sl = 0; sh.n_ch = 0; }
            __syncthreads();  // the tile may be zeroed again
            HOUGH_PT(6);
        }  // strips

        const int n_on = sh.n_on, n_pk = sh.n_peaks;
        if (give_up || n_pk > P.fPCAP) {
            if (tid == 0) P.deferred[atomicAdd(P.deferred_count, 1u)] = e;
            if (++overflow_run >= kGiveUpRun) { overflow_run = 0; skip_left = kGiveUpSkip; }
            continue;
        }
        overflow_run = 0;
        // the tile is dead: its first ONCAP words become the root tags
        for (int i = tid; i < n_on; i += nthr) if (HB(P, i, P.f_tile_bytes >> 2, 150)) roottag[i] = 0;

        // ---------------- S4: the K best peaks (key = (1023 - votes) << 22 | L, ascending)
        if (n_pk > P.K) {
            if (tid < 32) {  // threshold vote count c*: #(votes > c*) < K <= #(votes >= c*)
                int s = 0;
#pragma unroll
                for (int j = 0; j < 8; ++j) s += hist[255 - (lane * 8 + j)];  // descending votes
                int incl = s;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) { const int y = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += y; }
                int before = incl - s;
                if (before < P.K && P.K <= incl) {
                    int j = 0;
                    while (before + hist[255 - (lane * 8 + j)] < P.K) { before += hist[255 - (lane * 8 + j)]; ++j; }
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
            const int tcap = P.fSLCAP >> 1;  // tie list: keys in the first half of the strip list, peak positions in the second
            uint32_t* tie_key = slist;
            uint32_t* tie_pos = slist + tcap;
            for (int i0 = tid - lane; i0 < n_pk; i0 += nthr) {
                const int i = i0 + lane;
                uint32_t key = 0;
                int c = -1;
                if (i < n_pk) { key = peaks[i]; c = (int)(kCountMax - (key >> kLBits)); }
                const int a = warp_append(&sh.n_kept, c > cstar);
                if (c > cstar && HB(P, a, P.K, 151)) { kept[a] = key; kidx[a] = pidx[i]; }
                const int b = warp_append(&sh.n_ties, c == cstar);
                if (c == cstar && b < tcap && HB(P, b, tcap, 152)) { tie_key[b] = key; tie_pos[b] = (uint32_t)i; }
            }
            __syncthreads();
            const int n_ties = sh.n_ties, n_gt = sh.n_kept;
            if (n_ties > tcap) {
                if (tid == 0) P.deferred[atomicAdd(P.deferred_count, 1u)] = e;
                continue;
            }
            const int need = P.K - n_gt;  // 1 <= need <= n_ties: the `need` smallest keys among the ties
            for (int i = tid; i < n_ties; i += nthr) {
                const uint32_t key = tie_key[i];
                int rank = 0;
                for (int j = 0; j < n_ties; ++j) rank += (tie_key[j] < key);
                if (rank < need && HB(P, n_gt + rank, P.K, 153) && HB(P, tie_pos[i], P.fPCAP, 154)) { kept[n_gt + rank] = key; kidx[n_gt + rank] = pidx[tie_pos[i]]; }
            }
            if (tid == 0) sh.n_final = P.K;
        } else {
            for (int i = tid; i < n_pk; i += nthr) { kept[i] = peaks[i]; kidx[i] = pidx[i]; }
            if (tid == 0) sh.n_final = n_pk;
        }
        __syncthreads();
        const int n_kept = sh.n_final;
        for (int i = tid; i < n_kept; i += nthr) {  // slot = number of kept keys that are smaller (keys are unique)
            const uint32_t key = kept[i];
            int s = 0;
            for (int j = 0; j < n_kept; ++j) s += (kept[j] < key);
            if (HB(P, s, P.K, 155)) { sorted[s] = key; sidx[s] = kidx[i]; }
            ksize[i] = 0;
        }
        __syncthreads();
        HOUGH_PT(7);

        // ---------------- cluster of each kept peak: root, best-ranked kept peak of the same cluster, size
        for (int s = tid; s < n_kept; s += nthr) {
            const uint32_t root = suf_find(P, parent, (uint32_t)sidx[s]);
            kroot[s] = root;
            if (HB(P, root, n_on, 156)) atomicMax(roottag + root, (uint32_t)(P.K - s));  // the best-ranked (smallest slot) kept peak of the component wins
        }
        __syncthreads();
        HOUGH_PT(8);
        for (int i0 = tid - lane; i0 < n_on; i0 += nthr) {  // sizes of the components that own a kept peak
            const int i = i0 + lane;
            if (i < n_on) {
                const uint32_t id = roottag[suf_find(P, parent, (uint32_t)i)];
                if (id != 0 && HB(P, P.K - id, P.K, 157)) atomicAdd(ksize + (P.K - id), 1u);
            }
            __syncwarp();
        }
        __syncthreads();
        HOUGH_PT(10);

        // ---------------- records in rank order
        for (int s = tid; s < n_kept; s += nthr) {
            const uint32_t key = sorted[s];
            const uint32_t L = key & kLMask;
            const uint32_t c = kCountMax - (key >> kLBits);
            int rs = P.K - (int)roottag[kroot[s]];
            if (!HB(P, rs, n_kept, 158)) rs = 0;
            int t, r;
            split_L(P, L, t, r);
            const float th = theta_of_bin(P, t);
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
