// RFI clip kernels (PAPER.md:79 channel thresholding, PAPER.md:81 spectrum thresholding;
// thresholds per BASELINE.json north_star; readings B-i..B-ix in DESIGN.md section 3).
//
//   clip_channel_kernel   one CTA per (beam, channel) row: warp-shuffle reductions give the
//                         chunk sums (kept in shared memory) and the row's S, Q; the same CTA
//                         then thresholds, dilates and overwrites flagged chunks in place.
//   clip_spec_sum_kernel  column sums s_t over channels of the modified data (coalesced rows,
//                         channels split over the warps of a CTA, reduced through shared memory).
//   clip_spec_stats_kernel  one CTA per beam: M1, M2 -> mean_s, sig_s, threshold.
//   clip_spec_apply_kernel  flags spectra and overwrites flagged columns.
//
// Decisions are taken in fp64 with single IEEE operations in the oracle's order
// (__dadd_rn/__dmul_rn/__ddiv_rn/__dsqrt_rn are never contracted to FMA).  With uint8 input
// every sum is an exact integer, so masks are bit-reproducible; with float input the sums are
// fp64 in a different (tree) order and may differ from the oracle only within the guard band B-ix.
#include "mdsm_internal.h"

namespace {

constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;

template <typename T> struct Elem;
template <> struct Elem<float> {
    static constexpr int V = 4;
    using Vec = float4;
    using Acc = double;  // S, Q, chunk sums
    __device__ static void sums(const Vec &v, Acc &s, Acc &q)
    {
        double a = v.x, b = v.y, c = v.z, d = v.w;
        s = (a + b) + (c + d);
        q = fma(a, a, fma(b, b, fma(c, c, d * d)));
    }
};
template <> struct Elem<uint8_t> {
    static constexpr int V = 16;
    using Vec = uint4;
    using Acc = unsigned long long;
    __device__ static void sums(const Vec &v, Acc &s, Acc &q)
    {
        // four bytes per instruction: dp4a with ones gives the sum, with the word itself the sum of squares (exact in 32 bits)
        unsigned ss = 0, qq = 0;
        const unsigned w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            ss = __dp4a(w[i], 0x01010101u, ss);
            qq = __dp4a(w[i], w[i], qq);
        }
        s = ss;
        q = qq;
    }
};

template <typename A> __device__ __forceinline__ A shfl_xor(A v, int m);
template <> __device__ __forceinline__ double shfl_xor<double>(double v, int m) { return __shfl_xor_sync(0xffffffffu, v, m); }
template <> __device__ __forceinline__ unsigned long long shfl_xor<unsigned long long>(unsigned long long v, int m)
{
    return __shfl_xor_sync(0xffffffffu, v, m);
}

template <typename A> __device__ __forceinline__ A warp_sum(A v)
{
#pragma unroll
    for (int m = 16; m >= 1; m >>= 1) v += shfl_xor<A>(v, m);
    return v;
}

template <typename A> __device__ A block_sum(A v, A *red /*[kWarps]*/)
{
    v = warp_sum(v);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
    __syncthreads();
    A t = 0;
#pragma unroll
    for (int i = 0; i < kWarps; ++i) t += red[i];
    return t;
}

// mode 0: chunk = g lanes of one warp iteration (g power of two <= 32)
// mode 1: chunk = g/32 warp iterations of one warp (g % 32 == 0)
// mode 2: generic scalar path (any window, any alignment); chunk sums are recomputed from global
// STAGE 0: north_star's clip (statistics of the row itself); STAGE 1: the paper's bandpass stage (threshold on the chunk
// MEAN and replacement value come from the fit, chan_stats[b][c] = fit, threshold, -, (float)fit)
template <typename T, int MODE, int STAGE = 0>
__global__ void __launch_bounds__(kThreads)
clip_channel_kernel(T *__restrict__ in, int beam0, int nchans, long long nsamps, int window, double k_chan,
                    double *__restrict__ chan_stats, uint8_t *__restrict__ chan_mask)
{
    using E = Elem<T>;
    using Acc = typename E::Acc;
    constexpr int V = E::V;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const long long nchunk = nsamps / window;
    // layout: [csum: nchunk doubles (MODE<2 only)] [raw: nchunk bytes]
    double *csum = reinterpret_cast<double *>(smem_raw);
    uint8_t *raw = smem_raw + (MODE < 2 ? (size_t)nchunk * sizeof(double) : 0);
    __shared__ Acc red[kWarps];

    const int c = blockIdx.x;
    const int b = beam0 + blockIdx.y;
    T *row = in + ((size_t)b * nchans + c) * (size_t)nsamps;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    Acc S = 0, Q = 0;
    if (MODE == 0) {
        const int g = window / V;                              // a power of two <= 32 in this mode
        const int gshift = __ffs(g) - 1;
        const long long nvec = nsamps / V;
        const typename E::Vec *vrow = reinterpret_cast<const typename E::Vec *>(row);
        if (sizeof(T) == 4 && g >= 4) {
            // float rows: a thread takes FOUR consecutive vectors of a chunk, so that the fp64 shuffle tree over the chunk's
            // lanes is two levels shorter (the kernel is bound by instruction issue, not by memory)
            const int g4 = g >> 2;
            for (long long base = 0; base < nvec; base += 4LL * kThreads) {
                const long long i0 = base + 4LL * tid;
                Acc s = 0, q = 0;
                if (i0 < nvec) {                               // nvec is a multiple of g, g of 4: all four or none
                    typename E::Vec v[4];
#pragma unroll
                    for (int k = 0; k < 4; ++k) v[k] = vrow[i0 + k];
#pragma unroll
                    for (int k = 0; k < 4; ++k) {
                        Acc s1, q1;
                        E::sums(v[k], s1, q1);
                        s += s1;
                        q += q1;
                    }
                }
                S += s;
                Q += q;
                for (int m = 1; m < g4; m <<= 1) s += shfl_xor<Acc>(s, m);
                if (i0 < nvec && (lane & (g4 - 1)) == 0) csum[i0 >> gshift] = (double)s;
            }
        } else
        for (long long base = 0; base < nvec; base += kThreads) {
            const long long i = base + tid;
            Acc s = 0, q = 0;
            if (i < nvec) E::sums(vrow[i], s, q);
            S += s;
            Q += q;
            for (int m = 1; m < g; m <<= 1) s += shfl_xor<Acc>(s, m);
            if (i < nvec && (lane & (g - 1)) == 0) csum[i >> gshift] = (double)s;      // no 64-bit division in the loop
        }
    } else if (MODE == 1) {
        const int g = window / V;
        const typename E::Vec *vrow = reinterpret_cast<const typename E::Vec *>(row);
        for (long long j = warp; j < nchunk; j += kWarps) {
            Acc s = 0, q = 0;
            for (int k = lane; k < g; k += 32) {
                Acc s1, q1;
                E::sums(vrow[j * g + k], s1, q1);
                s += s1;
                q += q1;
            }
            S += s;
            Q += q;
            s = warp_sum(s);
            if (lane == 0) csum[j] = (double)s;
        }
    } else {
        for (long long t = tid; t < nsamps; t += kThreads) {
            Acc v = (Acc)row[t];
            S += v;
            Q += v * v;
        }
    }
    S = block_sum(S, red);
    Q = block_sum(Q, red);

    double thr_fit = 0.0;
    T repl_fit = 0;
    if (STAGE == 1) {
        const double *st = chan_stats + ((size_t)b * nchans + c) * 4;
        thr_fit = st[1];
        repl_fit = (T)st[3];
    }
    // B1: per-channel statistics, single IEEE ops in the oracle's order
    const double dN = (double)nsamps;
    const double mean = __ddiv_rn((double)S, dN);
    double var = __dsub_rn(__ddiv_rn((double)Q, dN), __dmul_rn(mean, mean));
    if (var < 0.0) var = 0.0;
    const double sig = __dsqrt_rn(var);
    const double thr = __dadd_rn(__dmul_rn((double)window, mean), __dmul_rn(__dmul_rn(k_chan, sig), __dsqrt_rn((double)window)));
    T repl;
    if (sizeof(T) == 1)
        repl = (T)(((unsigned long long)S + (unsigned long long)(nsamps / 2)) / (unsigned long long)nsamps);
    else
        repl = (T)mean;
    if (STAGE == 0 && tid == 0) {
        double *st = chan_stats + ((size_t)b * nchans + c) * 4;
        st[0] = mean; st[1] = sig; st[2] = thr; st[3] = (double)repl;
    }
    if (STAGE == 1) repl = repl_fit;

    // B2: raw flags
    for (long long j = tid; j < nchunk; j += kThreads) {
        double C;
        if (MODE < 2) {
            C = csum[j];
        } else {
            Acc s = 0;
            for (int k = 0; k < window; ++k) s += (Acc)row[j * window + k];
            C = (double)s;
        }
        raw[j] = (STAGE == 1 ? (__ddiv_rn(C, (double)window) > thr_fit) : (C > thr)) ? 1 : 0;
    }
    __syncthreads();
    // dilation by one chunk in time, mask output, in-place replacement
    uint8_t *mrow = chan_mask ? chan_mask + ((size_t)b * nchans + c) * (size_t)nchunk : nullptr;
    for (long long j = tid; j < nchunk; j += kThreads) {
        uint8_t m = raw[j];
        if (j > 0) m |= raw[j - 1];
        if (j + 1 < nchunk) m |= raw[j + 1];
        if (mrow) mrow[j] = m;
        if (m) {
            T *x = row + j * window;
            for (int k = 0; k < window; ++k) x[k] = repl;
        }
    }
}

// s_t = sum_c x[c][t] on the data as modified by the channel stage (B3, first half).
// CTA = 8 warps; covers 32*V consecutive samples; warp w adds channels c = w, w+8, ...
template <typename T, bool VEC>
__global__ void __launch_bounds__(kThreads)
clip_spec_sum_kernel(const T *__restrict__ in, int beam0, int nchans, long long nsamps, double *__restrict__ spec_sum)
{
    using E = Elem<T>;
    constexpr int V = VEC ? E::V : 1;
    using Acc = typename E::Acc;
    __shared__ Acc part[kWarps][32 * V + 1];
    const int b = beam0 + blockIdx.y;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const long long t0 = ((long long)blockIdx.x * 32 + lane) * V;
    const T *base = in + (size_t)b * nchans * (size_t)nsamps;
    Acc acc[V];
#pragma unroll
    for (int k = 0; k < V; ++k) acc[k] = 0;
    if (t0 < nsamps) {
        if (VEC) {
#pragma unroll 4
            for (int c = warp; c < nchans; c += kWarps) {
                const typename E::Vec v = *reinterpret_cast<const typename E::Vec *>(base + (size_t)c * nsamps + t0);
                if (sizeof(T) == 4) {
                    const float *f = reinterpret_cast<const float *>(&v);
#pragma unroll
                    for (int k = 0; k < V; ++k) acc[k] += (Acc)f[k];
                } else {
                    const unsigned *w = reinterpret_cast<const unsigned *>(&v);
#pragma unroll
                    for (int k = 0; k < V; ++k) acc[k] += (Acc)((w[k >> 2] >> (8 * (k & 3))) & 0xffu);
                }
            }
        } else {
            for (int c = warp; c < nchans; c += kWarps) acc[0] += (Acc)base[(size_t)c * nsamps + t0];
        }
    }
#pragma unroll
    for (int k = 0; k < V; ++k) part[warp][lane * V + k] = acc[k];
    __syncthreads();
    for (int i = threadIdx.x; i < 32 * V; i += kThreads) {
        Acc s = 0;
#pragma unroll
        for (int w = 0; w < kWarps; ++w) s += part[w][i];
        const long long t = (long long)blockIdx.x * 32 * V + i;
        if (t < nsamps) spec_sum[(size_t)b * nsamps + t] = (double)s;
    }
}

// One CTA per beam: M1 = sum s_t, M2 = sum s_t^2 -> spec_stats[b] = {thr, mean, sig}
template <bool IS_INT>
__global__ void __launch_bounds__(1024)
clip_spec_stats_kernel(const double *__restrict__ spec_sum, int beam0, long long nsamps, double k_spec,
                       double *__restrict__ spec_stats)
{
    const int b = beam0 + blockIdx.x;
    const double *s = spec_sum + (size_t)b * nsamps;
    __shared__ double rd[32][2];
    __shared__ unsigned long long ru[32][2];
    double m1 = 0.0, m2 = 0.0;
    unsigned long long u1 = 0, u2 = 0;
    for (long long t = threadIdx.x; t < nsamps; t += blockDim.x) {
        const double v = s[t];
        if (IS_INT) {
            const unsigned long long u = (unsigned long long)v;
            u1 += u;
            u2 += u * u;
        } else {
            m1 += v;
            m2 += v * v;
        }
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (IS_INT) {
        u1 = warp_sum(u1); u2 = warp_sum(u2);
        if (lane == 0) { ru[warp][0] = u1; ru[warp][1] = u2; }
    } else {
        m1 = warp_sum(m1); m2 = warp_sum(m2);
        if (lane == 0) { rd[warp][0] = m1; rd[warp][1] = m2; }
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double M1, M2;
        if (IS_INT) {
            unsigned long long a = 0, q = 0;
            for (int i = 0; i < (int)(blockDim.x >> 5); ++i) { a += ru[i][0]; q += ru[i][1]; }
            M1 = (double)a; M2 = (double)q;
        } else {
            M1 = 0.0; M2 = 0.0;
            for (int i = 0; i < (int)(blockDim.x >> 5); ++i) { M1 += rd[i][0]; M2 += rd[i][1]; }
        }
        const double dN = (double)nsamps;
        const double mean = __ddiv_rn(M1, dN);
        double var = __dsub_rn(__ddiv_rn(M2, dN), __dmul_rn(mean, mean));
        if (var < 0.0) var = 0.0;
        const double sig = __dsqrt_rn(var);
        spec_stats[4 * b + 0] = __dadd_rn(mean, __dmul_rn(k_spec, sig));
        spec_stats[4 * b + 1] = mean;
        spec_stats[4 * b + 2] = sig;
    }
}

// Thread = one time sample x kApplyChPer channels: a flagged spectrum is overwritten by nchans / kApplyChPer threads side by side.
constexpr int kApplyChPer = 128;
template <typename T>
__global__ void __launch_bounds__(kThreads)
clip_spec_apply_kernel(T *__restrict__ in, int beam0, int nchans, long long nsamps, const double *__restrict__ spec_sum,
                       const double *__restrict__ spec_stats, const double *__restrict__ chan_stats,
                       uint8_t *__restrict__ spec_mask)
{
    const int b = beam0 + blockIdx.z;
    const long long t = (long long)blockIdx.x * kThreads + threadIdx.x;
    if (t >= nsamps) return;
    const bool flag = spec_sum[(size_t)b * nsamps + t] > spec_stats[4 * b];
    if (blockIdx.y == 0 && spec_mask) spec_mask[(size_t)b * nsamps + t] = flag ? 1 : 0;
    if (flag) {
        const int c0 = blockIdx.y * kApplyChPer, c1 = min(nchans, c0 + kApplyChPer);
        T *col = in + ((size_t)b * nchans + c0) * (size_t)nsamps + t;
        const double *st = chan_stats + ((size_t)b * nchans + c0) * 4;
        for (int c = c0; c < c1; ++c, col += nsamps, st += 4) *col = (T)st[3];
    }
}

// ------------------------------------------------------------------ the paper's bandpass-fit stage
// PAPER.md:71-81, readings H-i..H-vii of DESIGN.md section 3; the oracle is orc_bandpass_clip_f32.  The paper fits the
// bandpass on the CPU between two kernels ("copied back to CPU memory"); here the fit is one small CTA
// per beam, so the whole stage stays asynchronous on the caller's stream:
//   bp_rowmean_kernel   H1: averaged bandpass bp[c] (one CTA per row, fp64)
//   bp_fit_kernel       H2-H4: median/MAD masking (bitonic sort in shared memory), neighbour interpolation, order-p
//                       normal equations (block reductions) solved by one thread, fit, rmse, mean/std of the bandpass
//   clip_channel_kernel<float, MODE, 1>   H5 with the fitted thresholds and replacement values
//   clip_spec_sum_kernel                  column sums of the modified data
//   bp_spec_apply_kernel  H6 + H7: spectrum flags, fitted-value replacement, bandpass subtraction
__global__ void __launch_bounds__(kThreads)
bp_rowmean_kernel(const float *__restrict__ in, int beam0, int nchans, long long nsamps, int vec, double *__restrict__ bp)
{
    __shared__ double red[kWarps];
    const int c = blockIdx.x, b = beam0 + blockIdx.y;
    const float *row = in + ((size_t)b * nchans + c) * (size_t)nsamps;
    double S = 0.0;
    if (vec) {
        const float4 *v = reinterpret_cast<const float4 *>(row);
        for (long long i = threadIdx.x; i < nsamps / 4; i += kThreads) {
            const float4 x = v[i];
            S += ((double)x.x + (double)x.y) + ((double)x.z + (double)x.w);
        }
    } else {
        for (long long t = threadIdx.x; t < nsamps; t += kThreads) S += (double)row[t];
    }
    S = block_sum(S, red);
    if (threadIdx.x == 0) bp[(size_t)b * nchans + c] = __ddiv_rn(S, (double)nsamps);
}

constexpr int kFitThreads = 1024;
constexpr int kFitMaxOrder = 12;

__device__ void bitonic_sort(double *a, int n /* power of two */)
{
    for (int k = 2; k <= n; k <<= 1)
        for (int j = k >> 1; j > 0; j >>= 1) {
            __syncthreads();
            for (int i = threadIdx.x; i < n; i += blockDim.x) {
                const int l = i ^ j;
                if (l > i) {
                    const double x = a[i], y = a[l];
                    const bool up = (i & k) == 0;
                    if ((x > y) == up) { a[i] = y; a[l] = x; }
                }
            }
        }
    __syncthreads();
}

__device__ double fit_block_sum(double v, double *red /*[32]*/)
{
    v = warp_sum(v);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
    __syncthreads();
    double t = 0.0;
    for (int i = 0; i < (int)(blockDim.x >> 5); ++i) t += red[i];
    return t;
}

// chan_stats[b][c][4] = fit, fit + k_chan*rmse (threshold on the chunk MEAN), interpolated bandpass, (double)(float)fit
// spec_stats[b][4]    = mean_bp + k_spec*std_bp, rmse, mean_bp, std_bp;  out_stats[b][4] = rmse, mean_bp, std_bp, masked channels
__global__ void __launch_bounds__(kFitThreads)
bp_fit_kernel(const double *__restrict__ bp_all, int beam0, int nchans, int npad, int order, double k_mask, double k_chan,
              double k_spec, double *__restrict__ chan_stats, double *__restrict__ spec_stats, double *__restrict__ out_fit,
              double *__restrict__ out_stats)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double *bp = reinterpret_cast<double *>(smem_raw);          // [nchans]
    double *srt = bp + nchans;                                  // [npad]
    double *bpi = srt + npad;                                   // [nchans]
    __shared__ double red[32];
    __shared__ double coef[kFitMaxOrder + 1];
    __shared__ double sums[3 * kFitMaxOrder + 2];
    __shared__ int s_nmask;
    const int b = beam0 + blockIdx.x, tid = threadIdx.x;
    const double inf = __longlong_as_double(0x7ff0000000000000LL);
    for (int c = tid; c < npad; c += kFitThreads) {
        const double v = c < nchans ? bp_all[(size_t)b * nchans + c] : inf;
        srt[c] = v;
        if (c < nchans) bp[c] = v;
    }
    if (tid == 0) s_nmask = 0;
    bitonic_sort(srt, npad);
    const double med = (nchans & 1) ? srt[nchans / 2] : __dmul_rn(0.5, __dadd_rn(srt[nchans / 2 - 1], srt[nchans / 2]));
    __syncthreads();
    for (int c = tid; c < npad; c += kFitThreads) srt[c] = c < nchans ? fabs(__dsub_rn(bp[c], med)) : inf;
    bitonic_sort(srt, npad);
    const double mad = (nchans & 1) ? srt[nchans / 2] : __dmul_rn(0.5, __dadd_rn(srt[nchans / 2 - 1], srt[nchans / 2]));
    const double lim = __dmul_rn(__dmul_rn(k_mask, 1.4826), mad);
    __syncthreads();
    // H2: mask + interpolate
    int nm = 0;
    for (int c = tid; c < nchans; c += kFitThreads) {
        double v = bp[c];
        if (__dsub_rn(v, med) > lim) {
            ++nm;
            int l = c - 1, r = c + 1;
            while (l >= 0 && __dsub_rn(bp[l], med) > lim) --l;
            while (r < nchans && __dsub_rn(bp[r], med) > lim) ++r;
            if (l >= 0 && r < nchans) v = __dmul_rn(0.5, __dadd_rn(bp[l], bp[r]));
            else if (l >= 0) v = bp[l];
            else if (r < nchans) v = bp[r];
        }
        bpi[c] = v;
    }
    if (nm) atomicAdd(&s_nmask, nm);
    __syncthreads();
    // H3: normal equations in u = 2c/(n-1) - 1: sums of u^k (k <= 2p) and of u^k y (k <= p)
    {
        double pu[2 * kFitMaxOrder + 1], py[kFitMaxOrder + 1];
        for (int k = 0; k <= 2 * order; ++k) pu[k] = 0.0;
        for (int k = 0; k <= order; ++k) py[k] = 0.0;
        for (int c = tid; c < nchans; c += kFitThreads) {
            const double u = nchans > 1 ? __dsub_rn(__ddiv_rn(__dmul_rn(2.0, (double)c), (double)(nchans - 1)), 1.0) : 0.0;
            double pw = 1.0;
            for (int k = 0; k <= 2 * order; ++k) {
                pu[k] += pw;
                if (k <= order) py[k] += pw * bpi[c];
                pw *= u;
            }
        }
        for (int k = 0; k <= 2 * order; ++k) { const double s = fit_block_sum(pu[k], red); if (tid == 0) sums[k] = s; }
        for (int k = 0; k <= order; ++k) { const double s = fit_block_sum(py[k], red); if (tid == 0) sums[2 * kFitMaxOrder + 1 + k] = s; }
    }
    __syncthreads();
    if (tid == 0) {
        double A[kFitMaxOrder + 1][kFitMaxOrder + 2];
        const int p = order;
        for (int i = 0; i <= p; ++i) {
            for (int j = 0; j <= p; ++j) A[i][j] = sums[i + j];
            A[i][p + 1] = sums[2 * kFitMaxOrder + 1 + i];
        }
        for (int i = 0; i <= p; ++i) {
            int piv = i;
            for (int r = i + 1; r <= p; ++r)
                if (fabs(A[r][i]) > fabs(A[piv][i])) piv = r;
            if (piv != i)
                for (int j = 0; j <= p + 1; ++j) { const double t = A[i][j]; A[i][j] = A[piv][j]; A[piv][j] = t; }
            for (int r = i + 1; r <= p; ++r) {
                const double f = A[r][i] / A[i][i];
                for (int j = i; j <= p + 1; ++j) A[r][j] = __dsub_rn(A[r][j], __dmul_rn(f, A[i][j]));
            }
        }
        for (int i = p; i >= 0; --i) {
            double s = A[i][p + 1];
            for (int j = i + 1; j <= p; ++j) s = __dsub_rn(s, __dmul_rn(A[i][j], coef[j]));
            coef[i] = s / A[i][i];
        }
    }
    __syncthreads();
    // fit (Horner) and H4
    double se = 0.0, s1 = 0.0, s2 = 0.0;
    for (int c = tid; c < nchans; c += kFitThreads) {
        const double u = nchans > 1 ? __dsub_rn(__ddiv_rn(__dmul_rn(2.0, (double)c), (double)(nchans - 1)), 1.0) : 0.0;
        double v = coef[order];
        for (int k = order - 1; k >= 0; --k) v = __dadd_rn(__dmul_rn(v, u), coef[k]);
        srt[c] = v;                                             // the fit, kept for the second loop (npad >= nchans)
        const double e = __dsub_rn(v, bpi[c]);
        se += e * e; s1 += bpi[c]; s2 += bpi[c] * bpi[c];
    }
    se = fit_block_sum(se, red);
    s1 = fit_block_sum(s1, red);
    s2 = fit_block_sum(s2, red);
    const double rmse = __dsqrt_rn(__ddiv_rn(se, (double)nchans));
    const double mean_bp = __ddiv_rn(s1, (double)nchans);
    double var_bp = __dsub_rn(__ddiv_rn(s2, (double)nchans), __dmul_rn(mean_bp, mean_bp));
    if (var_bp < 0.0) var_bp = 0.0;
    const double std_bp = __dsqrt_rn(var_bp);
    for (int c = tid; c < nchans; c += kFitThreads) {
        double *st = chan_stats + ((size_t)b * nchans + c) * 4;
        const double f = srt[c];
        st[0] = f; st[1] = __dadd_rn(f, __dmul_rn(k_chan, rmse)); st[2] = bpi[c]; st[3] = (double)(float)f;
        if (out_fit) { out_fit[((size_t)b * nchans + c) * 2] = f; out_fit[((size_t)b * nchans + c) * 2 + 1] = bpi[c]; }
    }
    if (tid == 0) {
        spec_stats[4 * b + 0] = __dadd_rn(mean_bp, __dmul_rn(k_spec, std_bp));
        spec_stats[4 * b + 1] = rmse; spec_stats[4 * b + 2] = mean_bp; spec_stats[4 * b + 3] = std_bp;
        if (out_stats) { out_stats[4 * b] = rmse; out_stats[4 * b + 1] = mean_bp; out_stats[4 * b + 2] = std_bp; out_stats[4 * b + 3] = (double)s_nmask; }
    }
}

// H6 + H7.  Thread = V consecutive time samples (V = 4: one 128-bit access, aligned rows; else 1) x kBpChPer channels.
constexpr int kBpChPer = 16;
template <int V>
__global__ void __launch_bounds__(kThreads)
bp_spec_apply_kernel(float *__restrict__ in, int beam0, int nchans, long long nsamps, const double *__restrict__ spec_sum,
                     const double *__restrict__ spec_stats, const double *__restrict__ chan_stats, int subtract,
                     uint8_t *__restrict__ spec_mask)
{
    const int b = beam0 + blockIdx.z;
    const long long t = ((long long)blockIdx.x * kThreads + threadIdx.x) * V;
    if (t >= nsamps) return;
    const double thr = spec_stats[4 * b];
    bool flag[V], any = false;
#pragma unroll
    for (int k = 0; k < V; ++k) {
        flag[k] = __ddiv_rn(spec_sum[(size_t)b * nsamps + t + k], (double)nchans) > thr;
        any |= flag[k];
        if (blockIdx.y == 0 && spec_mask) spec_mask[(size_t)b * nsamps + t + k] = flag[k] ? 1 : 0;
    }
    if (!any && !subtract) return;
    const int c0 = blockIdx.y * kBpChPer, c1 = min(nchans, c0 + kBpChPer);
    float *col = in + ((size_t)b * nchans + c0) * (size_t)nsamps + t;
    const double *st = chan_stats + ((size_t)b * nchans + c0) * 4;
    for (int c = c0; c < c1; ++c, col += nsamps, st += 4) {
        const float f = (float)st[3];
        if (V == 4) {
            float4 v = *reinterpret_cast<float4 *>(col);
            v.x = flag[0] ? f : v.x; v.y = flag[1] ? f : v.y; v.z = flag[2] ? f : v.z; v.w = flag[3] ? f : v.w;
            if (subtract) { v.x = v.x - f; v.y = v.y - f; v.z = v.z - f; v.w = v.w - f; }
            *reinterpret_cast<float4 *>(col) = v;
        } else {
            float v = flag[0] ? f : *col;
            if (subtract) v = v - f;
            *col = v;
        }
    }
}

template <typename T>
int launch_clip_t(mdsm_plan *p, T *in, int beam0, int nb, int window, double k_chan, double k_spec,
                  uint8_t *chan_mask, uint8_t *spec_mask, cudaStream_t st)
{
    constexpr int V = Elem<T>::V;
    const long long nsamps = p->nsamps;
    const long long nchunk = nsamps / window;
    const bool aligned = ((uintptr_t)in % 16 == 0) && (nsamps % V == 0);
    int mode = 2;
    if (aligned && window % V == 0) {
        const int g = window / V;
        if (g <= 32 && (g & (g - 1)) == 0) mode = 0;
        else if (g % 32 == 0) mode = 1;
    }
    size_t smem = (size_t)nchunk + (mode < 2 ? (size_t)nchunk * sizeof(double) : 0);
    if (mode < 2 && smem > 200 * 1024) { mode = 2; smem = (size_t)nchunk; }
    MDSM_REQUIRE(smem <= 200 * 1024, "nsamps/window = %lld chunks per channel exceeds the shared-memory flag buffer", nchunk);
    dim3 grid1(p->nchans, nb);
    auto k0 = clip_channel_kernel<T, 0>;
    auto k1 = clip_channel_kernel<T, 1>;
    auto k2 = clip_channel_kernel<T, 2>;
    auto kern = mode == 0 ? k0 : (mode == 1 ? k1 : k2);
    if (smem > 48 * 1024) MDSM_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    kern<<<grid1, kThreads, smem, st>>>(in, beam0, p->nchans, nsamps, window, k_chan, p->d_chan_stats, chan_mask);
    MDSM_CUDA_TRY(cudaGetLastError());

    double *spec_stats = p->d_spec_part;  // [nbeams][4]
    if (aligned) {
        dim3 grid2((unsigned)((nsamps + 32 * V - 1) / (32 * V)), nb);
        clip_spec_sum_kernel<T, true><<<grid2, kThreads, 0, st>>>(in, beam0, p->nchans, nsamps, p->d_spec_sum);
    } else {
        dim3 grid2((unsigned)((nsamps + 31) / 32), nb);
        clip_spec_sum_kernel<T, false><<<grid2, kThreads, 0, st>>>(in, beam0, p->nchans, nsamps, p->d_spec_sum);
    }
    MDSM_CUDA_TRY(cudaGetLastError());
    clip_spec_stats_kernel<sizeof(T) == 1><<<nb, 1024, 0, st>>>(p->d_spec_sum, beam0, nsamps, k_spec, spec_stats);
    MDSM_CUDA_TRY(cudaGetLastError());
    dim3 grid4((unsigned)((nsamps + kThreads - 1) / kThreads), (unsigned)((p->nchans + kApplyChPer - 1) / kApplyChPer), nb);
    MDSM_REQUIRE(grid4.y <= 65535 && nb <= 65535, "clip: grid too large");
    clip_spec_apply_kernel<T><<<grid4, kThreads, 0, st>>>(in, beam0, p->nchans, nsamps, p->d_spec_sum, spec_stats,
                                                          p->d_chan_stats, spec_mask);
    MDSM_CUDA_TRY(cudaGetLastError());
    p->launches += 4;
    return MDSM_OK;
}

}  // namespace

int mdsm_launch_clip(mdsm_plan *p, void *d_in, int dtype, int beam0, int nb, int window, double k_chan,
                     double k_spec, uint8_t *d_chan_mask, uint8_t *d_spec_mask, cudaStream_t st)
{
    if (dtype == MDSM_F32)
        return launch_clip_t<float>(p, (float *)d_in, beam0, nb, window, k_chan, k_spec, d_chan_mask, d_spec_mask, st);
    return launch_clip_t<uint8_t>(p, (uint8_t *)d_in, beam0, nb, window, k_chan, k_spec, d_chan_mask, d_spec_mask, st);
}

int mdsm_launch_bandpass_clip(mdsm_plan *p, float *in, int beam0, int nb, int window, int order, double k_mask, double k_chan,
                              double k_spec, int subtract, uint8_t *chan_mask, uint8_t *spec_mask, double *d_fit, double *d_stats,
                              cudaStream_t st)
{
    const long long nsamps = p->nsamps, nchunk = nsamps / window;
    const bool aligned = ((uintptr_t)in % 16 == 0) && (nsamps % 4 == 0);
    int npad = 1;
    while (npad < p->nchans) npad <<= 1;
    const size_t fit_smem = (size_t)(2 * p->nchans + npad) * sizeof(double);
    MDSM_REQUIRE(fit_smem <= 200 * 1024, "bandpass fit: nchans = %d exceeds the shared-memory sort buffer", p->nchans);
    dim3 grid1(p->nchans, nb);
    bp_rowmean_kernel<<<grid1, kThreads, 0, st>>>(in, beam0, p->nchans, nsamps, aligned ? 1 : 0, p->d_bandpass);
    MDSM_CUDA_TRY(cudaGetLastError());
    double *spec_stats = p->d_spec_part;
    if (fit_smem > 48 * 1024) MDSM_CUDA_TRY(cudaFuncSetAttribute(bp_fit_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fit_smem));
    bp_fit_kernel<<<nb, kFitThreads, fit_smem, st>>>(p->d_bandpass, beam0, p->nchans, npad, order, k_mask, k_chan, k_spec, p->d_chan_stats,
                                                    spec_stats, d_fit, d_stats);
    MDSM_CUDA_TRY(cudaGetLastError());
    int mode = 2;
    if (aligned && window % 4 == 0) {
        const int g = window / 4;
        if (g <= 32 && (g & (g - 1)) == 0) mode = 0;
        else if (g % 32 == 0) mode = 1;
    }
    size_t smem = (size_t)nchunk + (mode < 2 ? (size_t)nchunk * sizeof(double) : 0);
    if (mode < 2 && smem > 200 * 1024) { mode = 2; smem = (size_t)nchunk; }
    MDSM_REQUIRE(smem <= 200 * 1024, "nsamps/window = %lld chunks per channel exceeds the shared-memory flag buffer", nchunk);
    auto k0 = clip_channel_kernel<float, 0, 1>;
    auto k1 = clip_channel_kernel<float, 1, 1>;
    auto k2 = clip_channel_kernel<float, 2, 1>;
    auto kern = mode == 0 ? k0 : (mode == 1 ? k1 : k2);
    if (smem > 48 * 1024) MDSM_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    kern<<<grid1, kThreads, smem, st>>>(in, beam0, p->nchans, nsamps, window, k_chan, p->d_chan_stats, chan_mask);
    MDSM_CUDA_TRY(cudaGetLastError());
    if (aligned) {
        dim3 grid2((unsigned)((nsamps + 32 * 4 - 1) / (32 * 4)), nb);
        clip_spec_sum_kernel<float, true><<<grid2, kThreads, 0, st>>>(in, beam0, p->nchans, nsamps, p->d_spec_sum);
    } else {
        dim3 grid2((unsigned)((nsamps + 31) / 32), nb);
        clip_spec_sum_kernel<float, false><<<grid2, kThreads, 0, st>>>(in, beam0, p->nchans, nsamps, p->d_spec_sum);
    }
    MDSM_CUDA_TRY(cudaGetLastError());
    const int V = aligned ? 4 : 1;
    dim3 grid4((unsigned)((nsamps + (long long)kThreads * V - 1) / ((long long)kThreads * V)), (unsigned)((p->nchans + kBpChPer - 1) / kBpChPer), nb);
    MDSM_REQUIRE(grid4.y <= 65535 && nb <= 65535, "bandpass stage: grid too large");
    if (aligned)
        bp_spec_apply_kernel<4><<<grid4, kThreads, 0, st>>>(in, beam0, p->nchans, nsamps, p->d_spec_sum, spec_stats, p->d_chan_stats, subtract, spec_mask);
    else
        bp_spec_apply_kernel<1><<<grid4, kThreads, 0, st>>>(in, beam0, p->nchans, nsamps, p->d_spec_sum, spec_stats, p->d_chan_stats, subtract, spec_mask);
    MDSM_CUDA_TRY(cudaGetLastError());
    p->launches += 5;
    return MDSM_OK;
}
