// hough_track.cuh -- the stages around the Hough core (sm_100a): time slicing + phi = atan2(y, x) in front of it, line refit +
// "five consecutive planes" behind it.  Definitions: DESIGN.md Sec. 2 (O9-O12), readings B1-B6.
//
//   front end ("hits are divided into overlapping time windows of 10 ns, with a sliding step of 5 ns ...
//   (x, y, z) are transformed into the (phi, z) space"):
//     fe_count_kernel    one thread per RecoHit: validity, fixed-point time -> window range, integer CORDIC phi, window counts
//     fe_scan_kernel     one CTA: exclusive prefix sum of the window counts -> event offsets (int64) and write cursors
//     fe_scatter_kernel  one warp per fill, hits in input order, 32 at a time: every window a batch touches is filled in lane
//                        order, so a window's hits keep their input order (B4) without a sort and without atomics
//   back end (PAPER.md L106 seeds, L136 "continuous five vanes"):
//     hough_refit_kernel one CTA per event: exact 64-bit integer sums per kept candidate in shared memory (order independent),
//                        slope / intercept from one fixed sequence of double operations, plane mask -> longest run
#pragma once
#include "hough_kernels.cuh"

namespace hough {

// ---------------------------------------------------------------- front end
constexpr int kCordicIters = 20;   // residual rotation atan(2^-19) = 1.1e-4 degree
constexpr int kCordicGuard = 14;   // guard bits of the CORDIC state: |x_q| <= 2^15 keeps it inside int32
constexpr int kPhiFracBits = 16;   // phi LSB = 2^-16 degree (|phi_q| < 2^24: exact in fp32)
constexpr int kTimeFracBits = 8;   // time LSB = 2^-8 ns
constexpr int kXyFracBits = 6;     // x, y LSB = 2^-6 mm

struct FrontParams {
    int t0q, stepq, widthq;        // fixed-point window grid (2^-8 ns)
    int windows_per_fill;
    float xy_max;                  // rounded down to fp32
    int atan_q[kCordicIters];      // A_i = llround(atan(2^-i) 180 / pi 2^16)
    float* phi;                    // [max_hits] scratch: phi of every input hit
    int2* wrange;                  // [max_hits] scratch: (first window, last window) of every input hit; first > last = none
    int* counts;                   // [max_fills * windows_per_fill] hits per window
    long long* cursor;             // [max_fills * windows_per_fill] next write position of every window
    int* status;
};

// phi = atan2(y, x) in units of 2^-16 degree: integer CORDIC, vectoring mode (reading B2).  (xq, yq) != (0, 0), |xq|, |yq| <= 2^15.
__device__ __forceinline__ int cordic_phi_q(const FrontParams& FP, int xq, int yq)
{
    int X = abs(xq) << kCordicGuard, Y = yq * (1 << kCordicGuard), Z = 0;  // (a left shift of a negative value is undefined before C++20)
#pragma unroll
    for (int i = 0; i < kCordicIters; ++i) {
        const int xs = X >> i, ys = Y >> i;  // arithmetic shifts: floor
        if (Y >= 0) { X += ys; Y -= xs; Z += FP.atan_q[i]; }
        else { X -= ys; Y += xs; Z -= FP.atan_q[i]; }
    }
    const int half_turn = 180 << kPhiFracBits;
    if (xq >= 0) return Z;
    return yq >= 0 ? half_turn - Z : -half_turn - Z;
}

__device__ __forceinline__ long long floor_div(long long a, long long b)  // b > 0
{
    const long long q = a / b;
    return (a % b < 0) ? q - 1 : q;
}

__global__ void __launch_bounds__(256)
fe_count_kernel(const FrontParams FP, const float* __restrict__ x, const float* __restrict__ y, const float* __restrict__ z,
                const float* __restrict__ t, const long long* __restrict__ fill_offsets, int n_fills, long long n_hits)
{
    const float st = (float)(1 << kTimeFracBits), sx = (float)(1 << kXyFracBits);
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n_hits; i += (long long)gridDim.x * blockDim.x) {
        const float xf = __ldg(x + i), yf = __ldg(y + i), zf = __ldg(z + i), tf = __ldg(t + i);
        int2 wr = make_int2(0, -1);
        float phi = 0.f;
        // finite and in range (NaN fails every comparison; Inf exceeds the limits)
        const bool ok = (fabsf(xf) <= FP.xy_max) && (fabsf(yf) <= FP.xy_max) && (fabsf(zf) <= 3.402823466e+38f) &&
                        (fabsf(tf * st) < 2147483648.0f);
        if (ok) {
            const int xq = __float2int_rn(xf * sx), yq = __float2int_rn(yf * sx);  // exact products, ties to even
            // the fill that owns hit i: last f with fill_offsets[f] <= i
            int lo = 0, hi = n_fills - 1;
            while (lo < hi) { const int mid = (lo + hi + 1) >> 1; if (__ldg(fill_offsets + mid) <= i) lo = mid; else hi = mid - 1; }
            const bool in_fill = i >= __ldg(fill_offsets + lo) && i < __ldg(fill_offsets + lo + 1);
            if ((xq != 0 || yq != 0) && in_fill) {
                // window w holds the hit iff  w step <= d < w step + width  (64-bit: no overflow for any fp32 time)
                const long long d = (long long)__float2int_rn(tf * st) - (long long)FP.t0q;
                {
                    const long long w_hi64 = min(floor_div(d, FP.stepq), (long long)FP.windows_per_fill - 1);
                    const long long w_lo64 = max(floor_div(d - FP.widthq, FP.stepq) + 1, 0ll);
                    if (w_lo64 <= w_hi64) {
                        const int w_lo = (int)w_lo64, w_hi = (int)w_hi64;
                        wr = make_int2(w_lo, w_hi);
                        phi = (float)cordic_phi_q(FP, xq, yq) * (1.0f / (float)(1 << kPhiFracBits));  // exact: |phi_q| < 2^24
                        for (int w = w_lo; w <= w_hi; ++w) atomicAdd(FP.counts + (long long)lo * FP.windows_per_fill + w, 1);
                    }
                }
            }
        }
        FP.wrange[i] = wr;
        FP.phi[i] = phi;
    }
}

// Exclusive prefix sum of counts[n] -> offsets[n + 1] (int64) and cursor[n]; one CTA of 1024 threads, contiguous slices per thread.
__global__ void __launch_bounds__(1024)
fe_scan_kernel(const FrontParams FP, long long n, long long* __restrict__ offsets)
{
    __shared__ long long part[1024];
    const int tid = threadIdx.x;
    const long long per = (n + 1023) / 1024;
    const long long a = min((long long)tid * per, n), b = min(a + per, n);
    long long s = 0;
    for (long long i = a; i < b; ++i) s += FP.counts[i];
    part[tid] = s;
    __syncthreads();
    if (tid == 0) {
        long long run = 0;
        for (int k = 0; k < 1024; ++k) { const long long c = part[k]; part[k] = run; run += c; }
        offsets[n] = run;
    }
    __syncthreads();
    long long run = part[tid];
    for (long long i = a; i < b; ++i) { offsets[i] = run; FP.cursor[i] = run; run += FP.counts[i]; }
}

__global__ void __launch_bounds__(128)
fe_scatter_kernel(const FrontParams FP, const float* __restrict__ z, const long long* __restrict__ fill_offsets, int n_fills,
                  long long n_hits, float* __restrict__ u_out, float* __restrict__ v_out, int* __restrict__ src_out, long long capacity)
{
    const int lane = threadIdx.x & 31;
    const int warp = (int)((blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 5);
    const int n_warps = (int)(((long long)gridDim.x * blockDim.x) >> 5);
    const unsigned lt = (1u << lane) - 1u;
    for (int f = warp; f < n_fills; f += n_warps) {
        const long long a = fill_offsets[f], b = fill_offsets[f + 1];
        // fill offsets are caller data: a range outside [0, n_hits) would read window ranges that fe_count never wrote
        if (a < 0 || b < a || b > n_hits) { if (lane == 0) atomicOr(FP.status, 2); continue; }
        volatile long long* cur = FP.cursor + (long long)f * FP.windows_per_fill;  // written by lane 0, read by all lanes of this warp
        for (long long i0 = a; i0 < b; i0 += 32) {
            const long long i = i0 + lane;
            int nxt = 0x7fffffff, last = -1;
            float phi = 0.f, zz = 0.f;
            if (i < b) {
                const int2 wr = FP.wrange[i];
                if (wr.x <= wr.y) { nxt = wr.x; last = wr.y; phi = FP.phi[i]; zz = __ldg(z + i); }
            }
            while (true) {  // the windows this batch touches, in increasing order; inside one window the lanes keep their order
                int wmin = nxt;
#pragma unroll
                for (int o = 16; o; o >>= 1) wmin = min(wmin, __shfl_xor_sync(0xffffffffu, wmin, o));
                if (wmin == 0x7fffffff) break;  // warp-uniform
                const bool mine = (nxt == wmin);
                const unsigned m = __ballot_sync(0xffffffffu, mine);
                if (HB(FP, wmin, FP.windows_per_fill, 300)) {
                    const long long base = cur[wmin];
                    if (mine) {
                        const long long pos = base + __popc(m & lt);
                        if (pos < capacity) { u_out[pos] = phi; v_out[pos] = zz; src_out[pos] = (int)i; }
                        else atomicOr(FP.status, 8);
                    }
                    __syncwarp();  // every lane has read the cursor
                    if (lane == 0) cur[wmin] = base + __popc(m);
                    __syncwarp();  // ... and sees the new one in the next round
                }
                if (mine) nxt = (wmin < last) ? wmin + 1 : 0x7fffffff;
            }
        }
    }
}

// ---------------------------------------------------------------- back end: refit + found criterion
struct PlaneParams {
    int oq, pq;        // plane 0 and plane pitch in fixed-point hit units
    int n_planes, min_run, wrap;
};

struct Fit {  // mirrors hough_fit_t (32 bytes)
    int n_hits, max_run;
    unsigned long long plane_mask;
    float slope, intercept;
    int flags, reserved;
};

struct FitAcc {  // per kept candidate, in shared memory
    unsigned long long su, sv, suu, suv, mask;  // two's-complement sums of u_q, v_q, u_q^2, u_q v_q; plane bits
    unsigned int n, pad;
};

__device__ __forceinline__ int longest_run(unsigned long long m, int n_planes, int wrap)
{
    const unsigned long long full = n_planes >= 64 ? ~0ull : ((1ull << n_planes) - 1ull);
    m &= full;
    if (m == full) return n_planes;
    if (wrap) {  // rotate a clear bit to the top: then no run crosses the seam
        const int zb = __ffsll((long long)(~m & full)) - 1;  // a clear bit exists
        const int sh = zb + 1;
        if (sh < n_planes) m = ((m >> sh) | (m << (n_planes - sh))) & full;
    }
    int r = 0;
    while (m) { m &= m << 1; ++r; }
    return r;
}

__global__ void __launch_bounds__(256)
hough_refit_kernel(const DevParams P, const PlaneParams G, const float* __restrict__ u, const float* __restrict__ v,
                   const long long* __restrict__ offsets, int n_events, const int* __restrict__ n_found,
                   const int* __restrict__ labels, Fit* __restrict__ fits)
{
    HOUGH_DYNAMIC_SMEM(smem);
    FitAcc* acc = reinterpret_cast<FitAcc*>(smem);  // [K]
    const int tid = threadIdx.x, nthr = blockDim.x;
    for (int e = blockIdx.x; e < n_events; e += gridDim.x) {
        const long long g0 = offsets[e], g1 = offsets[e + 1];
        if (g0 < 0 || g1 < g0 || g1 > P.max_hits || (g1 - g0) > (long long)P.max_hits_per_event) continue;  // flagged by the find kernel: no records
        const int nk = min(max(n_found[e], 0), P.K);
        __syncthreads();  // the previous event's records are written
        for (int s = tid; s < nk; s += nthr) acc[s] = FitAcc{0ull, 0ull, 0ull, 0ull, 0ull, 0u, 0u};
        __syncthreads();
        for (long long i = g0 + tid; i < g1; i += nthr) {
            const int lab = labels[i];
            if (lab < 0 || lab >= nk) continue;  // unassigned or invalid hit; labels are caller data: one beyond the kept records is ignored
            const float uf = __ldg(u + i), vf = __ldg(v + i);
            // assign never labels an invalid hit; a caller's label on one is ignored (its coordinates would break the exactness bound)
            if (!(fabsf(uf) <= P.coord_max) || !(fabsf(vf) <= P.coord_max)) continue;
            const int uq = __float2int_rn(uf * P.hit_scale), vq = __float2int_rn(vf * P.hit_scale);
            FitAcc& A = acc[lab];
            atomicAdd(&A.n, 1u);
            atomicAdd(&A.su, (unsigned long long)(long long)uq);
            atomicAdd(&A.sv, (unsigned long long)(long long)vq);
            atomicAdd(&A.suu, (unsigned long long)((long long)uq * uq));
            atomicAdd(&A.suv, (unsigned long long)((long long)uq * vq));
            const long long num = 2ll * ((long long)uq - G.oq) + G.pq, den = 2ll * G.pq;
            long long pl = num / den;
            if (num % den < 0) --pl;  // floor
            if (pl >= 0 && pl < G.n_planes) atomicOr(&A.mask, 1ull << pl);
        }
        __syncthreads();
        for (int s = tid; s < nk; s += nthr) {
            const FitAcc A = acc[s];
            const long long n = (long long)A.n, su = (long long)A.su, sv = (long long)A.sv, suu = (long long)A.suu, suv = (long long)A.suv;
            const long long den = n * suu - su * su, num = n * suv - su * sv;  // exact: |u_q|, |v_q| <= 2^15, n < 2^16
            const int run = longest_run(A.mask, G.n_planes, G.wrap);
            int flags = run >= G.min_run ? 1 : 0;
            float slope = 0.f, icpt = 0.f;
            if (n < 2 || den == 0) {
                flags |= 2;
            } else {
                const double m = __ddiv_rn((double)num, (double)den);
                const double c = __ddiv_rn(__dadd_rn((double)sv, -__dmul_rn(m, (double)su)), (double)n);
                slope = (float)m;
                icpt = (float)__dmul_rn(c, 1.0 / (double)(1 << P.H));
            }
            int4* dst = reinterpret_cast<int4*>(fits + (size_t)e * P.K + s);
            dst[0] = make_int4((int)n, run, (int)(unsigned)(A.mask & 0xffffffffull), (int)(unsigned)(A.mask >> 32));
            dst[1] = make_int4(__float_as_int(slope), __float_as_int(icpt), flags, 0);
        }
    }
}

// ---------------------------------------------------------------- variant: iterative global-maximum peel-off (O13, reading B7)
//
// The paper's CPU peak rule ("a peak-finding algorithm identifies the bin with the highest number of
// entries ... track seeds are found by selecting the hits that align with the straight line"), repeated on the hits that
// remain.  One CTA per event; per track: the histogram of the remaining hits is refilled strip by strip (i32 counters in
// shared memory, S theta rows at a time), the maximum under the total order (count, -L) is kept across strips, its hits
// (|e| <= W_q) get the track's slot as label and leave the hit set.  labels[] doubles as the "removed" flag.  This variant
// is K times the work of the one-pass search and exists for comparison, not for throughput.
struct PeelShared {
    unsigned long long best;   // (count << 32) | (0xffffffff - L): larger = more votes, then lower linear index
    int removed, stop;
};

__global__ void __launch_bounds__(512)
hough_peel_kernel(const DevParams P, int S, const float* __restrict__ u, const float* __restrict__ v,
                  const long long* __restrict__ offsets, int n_events, Candidate* __restrict__ cands, int* __restrict__ n_found,
                  int* __restrict__ labels)
{
    HOUGH_DYNAMIC_SMEM(smem);
    __shared__ PeelShared sh;
    __shared__ unsigned long long wbest[16];
    int* tile = reinterpret_cast<int*>(smem);  // [S][n_rho]
    const int tid = threadIdx.x, nthr = blockDim.x, lane = tid & 31, warp = tid >> 5;
    const int half = P.F >= 1 ? (1 << (P.F - 1)) : 0;
    for (int e = blockIdx.x; e < n_events; e += gridDim.x) {
        const long long g0 = offsets[e], g1 = offsets[e + 1];
        __syncthreads();
        const bool bad_offsets = g0 < 0 || g1 < g0 || g1 > P.max_hits;
        if (bad_offsets || (g1 - g0) > (long long)P.max_hits_per_event) {
            if (tid == 0) { atomicOr(P.status, bad_offsets ? 2 : 1); n_found[e] = 0; }
            if (!bad_offsets) for (long long i = g0 + tid; i < g1; i += nthr) labels[i] = -1;
            continue;
        }
        const int ne = (int)(g1 - g0);
        for (int i = tid; i < ne; i += nthr) labels[g0 + i] = -1;
        int n_tracks = 0;
        while (n_tracks < P.K) {
            __syncthreads();  // labels of the previous track are written
            if (tid == 0) { sh.best = 0ull; sh.removed = 0; sh.stop = 0; }
            for (int base = 0; base < P.n_theta; base += S) {
                const int rows = min(S, P.n_theta - base);
                for (int i = tid; i < rows * P.n_rho; i += nthr) tile[i] = 0;
                __syncthreads();
                // one thread per (remaining hit, theta row of the strip)
                for (long long w = tid; w < (long long)ne * rows; w += nthr) {
                    const int h = (int)(w / rows), tl = (int)(w - (long long)h * rows);
                    if (labels[g0 + h] >= 0) continue;  // already on a track
                    const float uf = __ldg(u + g0 + h), vf = __ldg(v + g0 + h);
                    if (!(fabsf(uf) <= P.coord_max) || !(fabsf(vf) <= P.coord_max)) continue;
                    const int uq = __float2int_rn(uf * P.hit_scale), vq = __float2int_rn(vf * P.hit_scale);
                    const int a = uq * __ldg(P.Cq + base + tl) + (vq * __ldg(P.Sq + base + tl) + P.Oq);
                    const int r = a >> P.F;
                    if ((unsigned)r < (unsigned)P.n_rho && HB(P, tl * P.n_rho + r, S * P.n_rho, 320)) atomicAdd(&tile[tl * P.n_rho + r], 1);
                }
                __syncthreads();
                unsigned long long best = 0ull;
                for (int i = tid; i < rows * P.n_rho; i += nthr) {
                    const unsigned c = (unsigned)tile[i];
                    if (c) {
                        const unsigned L = (unsigned)(base * P.n_rho + i);  // i = tl * n_rho + r
                        const unsigned long long key = ((unsigned long long)c << 32) | (unsigned long long)(0xffffffffu - L);
                        if (key > best) best = key;
                    }
                }
#pragma unroll
                for (int o = 16; o; o >>= 1) { const unsigned long long y = __shfl_xor_sync(0xffffffffu, best, o); if (y > best) best = y; }
                if (lane == 0) wbest[warp] = best;
                __syncthreads();
                if (tid == 0) {
                    unsigned long long b = sh.best;
                    for (int k = 0; k < (nthr >> 5); ++k) if (wbest[k] > b) b = wbest[k];
                    sh.best = b;
                }
                __syncthreads();  // the tile may be cleared again
            }
            const unsigned long long best = sh.best;
            const int votes = (int)(best >> 32);
            if (votes < P.T) break;  // block-uniform: nothing above the threshold is left
            const unsigned L = 0xffffffffu - (unsigned)(best & 0xffffffffull);
            const int tb = (int)(L / (unsigned)P.n_rho), rb = (int)(L - (unsigned)tb * P.n_rho);
            const int Ct = __ldg(P.Cq + tb), St = __ldg(P.Sq + tb), Oc = P.Oq - (rb << P.F) - half;
            int mine = 0;
            for (int i = tid; i < ne; i += nthr) {
                if (labels[g0 + i] >= 0) continue;
                const float uf = __ldg(u + g0 + i), vf = __ldg(v + g0 + i);
                if (!(fabsf(uf) <= P.coord_max) || !(fabsf(vf) <= P.coord_max)) continue;
                const int uq = __float2int_rn(uf * P.hit_scale), vq = __float2int_rn(vf * P.hit_scale);
                const int ev = uq * Ct + (vq * St + Oc);
                if ((unsigned)abs(ev) <= (unsigned)P.Wq) { labels[g0 + i] = n_tracks; ++mine; }
            }
            if (mine) atomicAdd(&sh.removed, mine);
            __syncthreads();
            if (sh.removed == 0) break;  // a window narrower than half a bin missed every voter: no progress (B7)
            if (tid == 0) {
                const float th = theta_of_bin(P, tb);
                const float rho = (float)__dadd_rn(P.rho_min, __dmul_rn((double)rb + 0.5, P.d_rho));
                int4* dst = reinterpret_cast<int4*>(cands + (size_t)e * P.K + n_tracks);
                dst[0] = make_int4(tb, rb, votes, n_tracks);
                dst[1] = make_int4(0, __float_as_int(th), __float_as_int(rho), 0);
            }
            ++n_tracks;
        }
        if (tid == 0) n_found[e] = n_tracks;
    }
}

// ---------------------------------------------------------------- variant: two-stage (coarse -> fine) Hough (O14, reading B8)
//
// The paper's own answer to the shared-memory limit (Fig. 5: "a coarse-binning histogram followed by a
// fine-binning histogram").  One CTA per event: coarse histogram (c_theta x c_rho fine bins per coarse bin, one theta row per
// coarse row) -> coarse local maxima -> best K -> per kept coarse peak a fine patch of 3 x 3 coarse bins filled exactly,
// its maximum is the candidate; duplicates merged, ranked by (votes desc, linear index asc).
struct TwoStageParams {
    int c_theta, c_rho, nT, nR;   // coarse factors and coarse grid
    int cp_cap;                   // capacity of the coarse-peak list: ceil(nT / 2) * ceil(nR / 2) (no two strict maxima touch)
    int off_patch, off_cpeaks, off_ckept, off_fkeys;  // byte offsets into dynamic shared memory (the coarse tile starts at 0)
};

struct TwoStageShared {
    int n_cp, n_f;
    unsigned long long best;
};

__device__ __forceinline__ bool ts_hit(const DevParams& P, const float* __restrict__ u, const float* __restrict__ v, long long i, int& uq, int& vq)
{
    const float uf = __ldg(u + i), vf = __ldg(v + i);
    if (!(fabsf(uf) <= P.coord_max) || !(fabsf(vf) <= P.coord_max)) return false;
    uq = __float2int_rn(uf * P.hit_scale);
    vq = __float2int_rn(vf * P.hit_scale);
    return true;
}

__global__ void __launch_bounds__(512)
hough_two_stage_kernel(const DevParams P, const TwoStageParams Q, const float* __restrict__ u, const float* __restrict__ v,
                       const long long* __restrict__ offsets, int n_events, Candidate* __restrict__ cands, int* __restrict__ n_found)
{
    HOUGH_DYNAMIC_SMEM(smem);
    __shared__ TwoStageShared sh;
    __shared__ unsigned long long wbest[16];
    int* coarse = reinterpret_cast<int*>(smem);                                                    // [nT][nR]
    int* patch = reinterpret_cast<int*>(smem + Q.off_patch);                                       // [3 c_theta][3 c_rho]
    unsigned long long* cpeaks = reinterpret_cast<unsigned long long*>(smem + Q.off_cpeaks);       // [cp_cap]
    unsigned long long* ckept = reinterpret_cast<unsigned long long*>(smem + Q.off_ckept);         // [K]
    unsigned long long* fkeys = reinterpret_cast<unsigned long long*>(smem + Q.off_fkeys);         // [K]
    const int tid = threadIdx.x, nthr = blockDim.x, lane = tid & 31, warp = tid >> 5;
    const int n_cbins = Q.nT * Q.nR;
    for (int e = blockIdx.x; e < n_events; e += gridDim.x) {
        const long long g0 = offsets[e], g1 = offsets[e + 1];
        __syncthreads();
        const bool bad_offsets = g0 < 0 || g1 < g0 || g1 > P.max_hits;
        if (bad_offsets || (g1 - g0) > (long long)P.max_hits_per_event) {
            if (tid == 0) { atomicOr(P.status, bad_offsets ? 2 : 1); n_found[e] = 0; }
            continue;
        }
        const int ne = (int)(g1 - g0);
        if (tid == 0) { sh.n_cp = 0; sh.n_f = 0; }
        for (int i = tid; i < n_cbins; i += nthr) coarse[i] = 0;
        __syncthreads();
        // ---- stage 1: coarse histogram, one thread per (hit, coarse row)
        for (long long w = tid; w < (long long)ne * Q.nT; w += nthr) {
            const int h = (int)(w / Q.nT), T = (int)(w - (long long)h * Q.nT);
            int uq, vq;
            if (!ts_hit(P, u, v, g0 + h, uq, vq)) continue;
            const int t = min(T * Q.c_theta + Q.c_theta / 2, P.n_theta - 1);
            const int r = (uq * __ldg(P.Cq + t) + (vq * __ldg(P.Sq + t) + P.Oq)) >> P.F;
            if ((unsigned)r < (unsigned)P.n_rho && HB(P, T * Q.nR + r / Q.c_rho, n_cbins, 330)) atomicAdd(&coarse[T * Q.nR + r / Q.c_rho], 1);
        }
        __syncthreads();
        // ---- coarse peaks: strict local maxima >= T under (count, -index)
        for (int i = tid; i < n_cbins; i += nthr) {
            const int c = coarse[i];
            if (c < P.T) continue;
            const int T = i / Q.nR, R = i - T * Q.nR;
            bool pk = true;
            for (int dT = -1; dT <= 1 && pk; ++dT)
                for (int dR = -1; dR <= 1; ++dR) {
                    if (!dT && !dR) continue;
                    const int TT = T + dT, RR = R + dR;
                    if (TT < 0 || TT >= Q.nT || RR < 0 || RR >= Q.nR) continue;
                    const int j = TT * Q.nR + RR, cj = coarse[j];
                    if (cj > c || (cj == c && j < i)) { pk = false; break; }
                }
            if (pk) {
                const int k = atomicAdd(&sh.n_cp, 1);
                if (HB(P, k, Q.cp_cap, 331)) cpeaks[k] = ((unsigned long long)(unsigned)c << 32) | (unsigned long long)(0xffffffffu - (unsigned)i);
            }
        }
        __syncthreads();
        const int n_cp = min(sh.n_cp, Q.cp_cap), n_ck = min(n_cp, P.K);
        for (int i = tid; i < n_cp; i += nthr) {  // rank by counting (keys are unique): the K largest keys, best first
            const unsigned long long key = cpeaks[i];
            int rank = 0;
            for (int j = 0; j < n_cp; ++j) rank += (cpeaks[j] > key);
            if (rank < P.K) ckept[rank] = key;
        }
        __syncthreads();
        // ---- stage 2: one exact fine patch per kept coarse peak
        const int PR = 3 * Q.c_rho;
        for (int s = 0; s < n_ck; ++s) {
            const unsigned ci = 0xffffffffu - (unsigned)(ckept[s] & 0xffffffffull);
            const int T = (int)(ci / (unsigned)Q.nR), R = (int)(ci - (unsigned)T * Q.nR);
            const int t0 = max(0, (T - 1) * Q.c_theta), t1 = min(P.n_theta, (T + 2) * Q.c_theta);
            const int r0 = max(0, (R - 1) * Q.c_rho), r1 = min(P.n_rho, (R + 2) * Q.c_rho);
            const int rows = t1 - t0;
            for (int i = tid; i < 3 * Q.c_theta * PR; i += nthr) patch[i] = 0;
            __syncthreads();
            for (long long w = tid; w < (long long)ne * rows; w += nthr) {
                const int h = (int)(w / rows), t = t0 + (int)(w - (long long)h * rows);
                int uq, vq;
                if (!ts_hit(P, u, v, g0 + h, uq, vq)) continue;
                const int r = (uq * __ldg(P.Cq + t) + (vq * __ldg(P.Sq + t) + P.Oq)) >> P.F;
                if (r >= r0 && r < r1 && HB(P, (t - t0) * PR + (r - r0), 3 * Q.c_theta * PR, 332)) atomicAdd(&patch[(t - t0) * PR + (r - r0)], 1);
            }
            __syncthreads();
            unsigned long long best = 0ull;
            for (int i = tid; i < rows * PR; i += nthr) {
                const int tl = i / PR, rl = i - tl * PR;
                const unsigned c = (unsigned)patch[i];
                if (c && r0 + rl < r1) {
                    const unsigned L = (unsigned)((t0 + tl) * P.n_rho + r0 + rl);
                    const unsigned long long key = ((unsigned long long)c << 32) | (unsigned long long)(0xffffffffu - L);
                    if (key > best) best = key;
                }
            }
#pragma unroll
            for (int o = 16; o; o >>= 1) { const unsigned long long y = __shfl_xor_sync(0xffffffffu, best, o); if (y > best) best = y; }
            if (lane == 0) wbest[warp] = best;
            __syncthreads();
            if (tid == 0) {
                unsigned long long b = 0ull;
                for (int k = 0; k < (nthr >> 5); ++k) if (wbest[k] > b) b = wbest[k];
                if ((int)(b >> 32) >= P.T) fkeys[sh.n_f++] = b;
            }
            __syncthreads();  // the patch may be cleared again
        }
        // ---- merge duplicates, rank (votes desc, linear index asc), write the records
        const int n_f = sh.n_f;
        for (int i = tid; i < n_f; i += nthr) {
            const unsigned long long key = fkeys[i];
            bool dup = false;
            for (int j = 0; j < i; ++j) dup |= (fkeys[j] == key);
            if (dup) continue;
            int rank = 0;
            for (int j = 0; j < n_f; ++j) {
                if (fkeys[j] > key) {  // count every distinct larger key once: at its first occurrence
                    bool first = true;
                    for (int q = 0; q < j; ++q) first &= (fkeys[q] != fkeys[j]);
                    rank += first;
                }
            }
            const unsigned L = 0xffffffffu - (unsigned)(key & 0xffffffffull);
            const int t = (int)(L / (unsigned)P.n_rho), r = (int)(L - (unsigned)t * P.n_rho);
            const float th = theta_of_bin(P, t);
            const float rho = (float)__dadd_rn(P.rho_min, __dmul_rn((double)r + 0.5, P.d_rho));
            int4* dst = reinterpret_cast<int4*>(cands + (size_t)e * P.K + rank);
            dst[0] = make_int4(t, r, (int)(key >> 32), rank);
            dst[1] = make_int4(0, __float_as_int(th), __float_as_int(rho), 0);
        }
        __syncthreads();
        if (tid == 0) {
            int distinct = 0;
            for (int i = 0; i < n_f; ++i) {
                bool dup = false;
                for (int j = 0; j < i; ++j) dup |= (fkeys[j] == fkeys[i]);
                distinct += !dup;
            }
            n_found[e] = distinct;
        }
    }
}

}  // namespace hough
