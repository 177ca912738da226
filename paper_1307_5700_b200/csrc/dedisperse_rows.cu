// Brute-force dedispersion for sm_100a as "exact channel-group pre-sums + a sum of shifted rows"
// (BASELINE.json north_star item 2).
//
//   out[b][d][t] = sum_c in[b][c][t + delay(d,c)]
//
// Step 1, pre-pass (group_presum_*_kernel).  The channels are cut into groups of G adjacent channels
// (c0 .. c0+G-1).  Inside a group the delays RELATIVE to its first channel,
//   delta_i(d) = delay(d, c0+i) - delay(d, c0),   i = 1 .. G-1,
// take only a few distinct values over the whole DM grid (cfg 3, G = 4: 5.7 patterns per channel on average),
// because adjacent channels' delays differ by a few samples at most.  For every (group, pattern) the pre-pass
// writes ONE row of plan scratch
//   y[(g, pattern)][t] = sum_i in[c0+i][t + delta_i]
// so that   out[d][t] = sum_g y[(g, pattern(d,g))][t + delay(d, c0_g)]:
// exactly the same terms as the definition, added G at a time (uint8: bit-exact; fp32: another summation order,
// inside the tolerance).  The main kernel then needs nchans/G adds and operand words per output instead of nchans.
//
// Step 2, main kernel (dedisperse_rows_kernel).  Persistent CTAs (one per SM) walk tiles = one beam x DB = NW*D
// consecutive DM trials x `span` output samples.  A producer warp streams SLABS -- the y rows that the Q channel
// groups of the slab need for this DM block, each row starting at its own 16-byte-aligned, delay-dependent sample --
// into a ring of shared-memory stages with 1-D TMA bulk copies (cp.async.bulk ... mbarrier::complete_tx), together
// with the slab's slice of the ENTRY table (one shared-memory byte offset per (DM, group)).  A consumer warp owns D DM
// trials; lane l owns the outputs t0 + l + 32 i (i < T) of each of them (fp32) and adds, per (DM, group), the T words
// at entry + 4 l + 128 i: conflict-free 32-bit shared-memory loads at ANY delay (no alignment cases, no register-offset
// dispatch, no branches in the loop).  The kernel is bound by the shared-memory pipe at one operand word per add;
// pre-summing is what makes a word worth G algorithmic adds.
//   uint8: y holds uint16 group sums (G*255 < 2^16); a thread's accumulators are packed u16x2 lanes, one 32-bit
//   shared-memory word = two samples.  A group whose offset is ODD relative to the word grid would need its words
//   shifted by one lane; instead every DM keeps an even-phase row E (word k = outputs 2k, 2k+1) and an odd-phase row
//   O (word k = outputs 2k-1, 2k) and both add the words as loaded; the rows are merged (one lane shuffle) when a
//   PART of <= 256 channels (the most a 16-bit lane holds) is flushed into the uint32 output.
// The time axis of a tile is SHEARED: DM dl of a block owns outputs [tile_t0 - sigma_dl, +span) with sigma_dl ~ half
// the band-edge delay slope, which halves the length of the staged rows.
#include <algorithm>
#include <array>
#include <cmath>
#include <map>
#include <vector>

#include "mdsm_internal.h"

namespace {

// ------------------------------------------------------------------ PTX helpers
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("{ .reg .b64 t; mbarrier.arrive.shared::cta.b64 t, [%0]; }" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("{ .reg .b64 t; mbarrier.arrive.expect_tx.shared::cta.b64 t, [%0], %1; }" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t *bar, uint32_t parity)
{
    uint32_t done;
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t"
        "}" : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    return done != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    while (!mbar_try_wait(bar, parity)) {}
}
// the producer runs several stages ahead, so it sleeps between polls instead of taking issue slots
__device__ __forceinline__ void mbar_wait_sleep(uint64_t *bar, uint32_t parity)
{
    while (!mbar_try_wait(bar, parity)) __nanosleep(200);
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst_smem),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// ------------------------------------------------------------------ step 1: the pre-pass
constexpr int kGMax = 8;              // largest channel group
constexpr int kPreThreads = 256;
constexpr int kPreChunkF32 = 2048;    // samples of a y row per CTA (fp32): 8 per thread
constexpr int kPreChunkU8 = 4096;     // uint8: 16 per thread, four at a time

struct PreArgs {
    const void *in;
    void *y;
    const int32_t *group_row0;        // [ngroups + 1] first y row of a group
    const int16_t *ydelta;            // [nyrows][kGMax] delay of channel c0 + i relative to channel c0
    int beam0, nslots, nchans, G, nyrows, dmax;
    int delta_off;                    // byte offset of the group's pattern table inside the dynamic shared memory
    long long nsamps, ystride;
};

// fp32: one CTA = one channel group x one chunk of kPreChunkF32 samples x one beam.  The G raw rows of the chunk (plus
// the largest delta) go to shared memory once and serve every pattern of the group; thread `tid` owns the samples
// tid + 256 k, so that the shifted reads are conflict-free at any delta and the y stores are coalesced.
// TIn/TOut = float/float (MDSM_F32) or uint16/uint32 (MDSM_U16: the same 32-bit rows with integer sums).
template <int G, typename TIn, typename TOut>
__global__ void __launch_bounds__(kPreThreads) group_presum_w32_kernel(const PreArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    TOut *sm = reinterpret_cast<TOut *>(smem_raw);
    const int g = blockIdx.y, b = a.beam0 + blockIdx.z;
    const int c0 = g * a.G;
    const long long t0 = (long long)blockIdx.x * kPreChunkF32;
    const int pitch = kPreChunkF32 + a.dmax;
    const TIn *in = reinterpret_cast<const TIn *>(a.in) + (size_t)b * a.nchans * (size_t)a.nsamps;
#pragma unroll
    for (int i = 0; i < G; ++i) {
        const bool have = c0 + i < a.nchans;
        const TIn *row = in + (size_t)(have ? c0 + i : 0) * a.nsamps;
        for (int s = threadIdx.x; s < pitch; s += kPreThreads) sm[i * pitch + s] = (have && t0 + s < a.nsamps) ? (TOut)row[t0 + s] : (TOut)0;
    }
    // the group's patterns go to shared memory too: the loop below must not wait on L2 for its next deltas
    const int row0 = a.group_row0[g], row1 = a.group_row0[g + 1];
    int16_t *sdelta = reinterpret_cast<int16_t *>(smem_raw + a.delta_off);
    for (int k = threadIdx.x; k < (row1 - row0) * kGMax; k += kPreThreads) sdelta[k] = a.ydelta[(size_t)row0 * kGMax + k];
    __syncthreads();
    TOut *ybeam = reinterpret_cast<TOut *>(a.y) + (size_t)(b % a.nslots) * a.nyrows * (size_t)a.ystride;
    TOut x0[kPreChunkF32 / kPreThreads];                         // delta_0 = 0 for every pattern: the first channel stays in registers
#pragma unroll
    for (int k = 0; k < kPreChunkF32 / kPreThreads; ++k) x0[k] = sm[threadIdx.x + k * kPreThreads];
    for (int r = row0; r < row1; ++r) {
        int dl[G];
#pragma unroll
        for (int i = 0; i < G; ++i) dl[i] = sdelta[(r - row0) * kGMax + i];
        TOut *yrow = ybeam + (size_t)r * a.ystride + t0;
        TOut v[kPreChunkF32 / kPreThreads];
#pragma unroll
        for (int k = 0; k < kPreChunkF32 / kPreThreads; ++k) {
            const int s = threadIdx.x + k * kPreThreads;
            TOut acc = x0[k];
#pragma unroll
            for (int i = 1; i < G; ++i) acc += sm[i * pitch + s + dl[i]];
            v[k] = acc;
        }
#pragma unroll
        for (int k = 0; k < kPreChunkF32 / kPreThreads; ++k) {
            const int s = threadIdx.x + k * kPreThreads;
            if (t0 + s < a.ystride) yrow[s] = v[k];
        }
    }
}

// uint8 -> uint16 group sums.  Raw rows are kept as bytes; thread `tid` owns the samples 4 (tid + 256 k) .. +3: the four
// bytes of row i at delta_i come out of two aligned words with one funnel shift (the shift is the same for the whole
// row), are spread to two u16x2 words and added lane-wise; one 8-byte store per thread.
template <int G>
__global__ void __launch_bounds__(kPreThreads) group_presum_u8_kernel(const PreArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int g = blockIdx.y, b = a.beam0 + blockIdx.z;
    const int c0 = g * a.G;
    const long long t0 = (long long)blockIdx.x * kPreChunkU8;
    const int pitch = kPreChunkU8 + ((a.dmax + 3) & ~3) + 4;          // bytes, whole words, one spare word
    const uint8_t *in = reinterpret_cast<const uint8_t *>(a.in) + (size_t)b * a.nchans * (size_t)a.nsamps;
#pragma unroll
    for (int i = 0; i < G; ++i) {
        const bool have = c0 + i < a.nchans;
        const uint8_t *row = in + (size_t)(have ? c0 + i : 0) * a.nsamps;
        if ((((uintptr_t)(row + t0)) & 3) == 0) {
            for (int s = threadIdx.x * 4; s < pitch; s += kPreThreads * 4) {
                uint32_t w = 0;
                if (have) {
                    if (t0 + s + 3 < a.nsamps) w = *reinterpret_cast<const uint32_t *>(row + t0 + s);
                    else
                        for (int k = 0; k < 4; ++k)
                            if (t0 + s + k < a.nsamps) w |= (uint32_t)row[t0 + s + k] << (8 * k);
                }
                *reinterpret_cast<uint32_t *>(smem_raw + i * pitch + s) = w;
            }
        } else {
            for (int s = threadIdx.x; s < pitch; s += kPreThreads) smem_raw[i * pitch + s] = (have && t0 + s < a.nsamps) ? row[t0 + s] : (uint8_t)0;
        }
    }
    const int row0 = a.group_row0[g], row1 = a.group_row0[g + 1];
    int16_t *sdelta = reinterpret_cast<int16_t *>(smem_raw + a.delta_off);
    for (int k = threadIdx.x; k < (row1 - row0) * kGMax; k += kPreThreads) sdelta[k] = a.ydelta[(size_t)row0 * kGMax + k];
    __syncthreads();
    uint16_t *ybeam = reinterpret_cast<uint16_t *>(a.y) + (size_t)(b % a.nslots) * a.nyrows * (size_t)a.ystride;
    for (int r = row0; r < row1; ++r) {
        int dl[G];
#pragma unroll
        for (int i = 0; i < G; ++i) dl[i] = sdelta[(r - row0) * kGMax + i];
        uint16_t *yrow = ybeam + (size_t)r * a.ystride + t0;
#pragma unroll
        for (int k = 0; k < kPreChunkU8 / (4 * kPreThreads); ++k) {
            const int s = 4 * (threadIdx.x + k * kPreThreads);
            uint32_t lo = 0, hi = 0;
#pragma unroll
            for (int i = 0; i < G; ++i) {
                const uint32_t *w = reinterpret_cast<const uint32_t *>(smem_raw + i * pitch + ((s + dl[i]) & ~3));
                const uint32_t v = __funnelshift_r(w[0], w[1], 8 * (dl[i] & 3));
                lo += __byte_perm(v, 0, 0x4140);
                hi += __byte_perm(v, 0, 0x4342);
            }
            if (t0 + s < a.ystride) *reinterpret_cast<uint2 *>(yrow + s) = make_uint2(lo, hi);      // ystride % 8 == 0
        }
    }
}


// 4-bit samples (two per byte along time, low nibble first) -> uint16 group sums.  Thread `tid` owns the samples
// 4 (tid + 256 k) .. +3: the four nibbles of row i at delta_i are 16 bits starting at nibble s + delta_i, cut out of two
// aligned words with one funnel shift and spread to two u16x2 words.
template <int G>
__global__ void __launch_bounds__(kPreThreads) group_presum_u4_kernel(const PreArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int g = blockIdx.y, b = a.beam0 + blockIdx.z;
    const int c0 = g * a.G;
    const long long t0 = (long long)blockIdx.x * kPreChunkU8;                   // samples; t0 / 2 bytes into the row
    const int pitch = (((kPreChunkU8 + a.dmax) / 2 + 3) & ~3) + 8;               // bytes, whole words, room for the two-word fetch
    const long long row_bytes = a.nsamps / 2;
    const uint8_t *in = reinterpret_cast<const uint8_t *>(a.in) + (size_t)b * a.nchans * (size_t)row_bytes;
#pragma unroll
    for (int i = 0; i < G; ++i) {
        const bool have = c0 + i < a.nchans;
        const uint8_t *row = in + (size_t)(have ? c0 + i : 0) * row_bytes;
        for (int s = threadIdx.x; s < pitch; s += kPreThreads) smem_raw[i * pitch + s] = (have && t0 / 2 + s < row_bytes) ? row[t0 / 2 + s] : (uint8_t)0;
    }
    const int row0 = a.group_row0[g], row1 = a.group_row0[g + 1];
    int16_t *sdelta = reinterpret_cast<int16_t *>(smem_raw + a.delta_off);
    for (int k = threadIdx.x; k < (row1 - row0) * kGMax; k += kPreThreads) sdelta[k] = a.ydelta[(size_t)row0 * kGMax + k];
    __syncthreads();
    uint16_t *ybeam = reinterpret_cast<uint16_t *>(a.y) + (size_t)(b % a.nslots) * a.nyrows * (size_t)a.ystride;
    for (int r = row0; r < row1; ++r) {
        int dl[G];
#pragma unroll
        for (int i = 0; i < G; ++i) dl[i] = sdelta[(r - row0) * kGMax + i];
        uint16_t *yrow = ybeam + (size_t)r * a.ystride + t0;
#pragma unroll
        for (int k = 0; k < kPreChunkU8 / (4 * kPreThreads); ++k) {
            const int s = 4 * (threadIdx.x + k * kPreThreads);
            uint32_t lo = 0, hi = 0;
#pragma unroll
            for (int i = 0; i < G; ++i) {
                const int nib = s + dl[i];                                      // first nibble of the four
                const uint32_t *w = reinterpret_cast<const uint32_t *>(smem_raw + i * pitch + ((nib >> 1) & ~3));
                const uint32_t v = __funnelshift_r(w[0], w[1], 4 * (nib & 7));
                lo += (v & 0xfu) | ((v & 0xf0u) << 12);
                hi += ((v >> 8) & 0xfu) | ((v & 0xf000u) << 4);
            }
            if (t0 + s < a.ystride) *reinterpret_cast<uint2 *>(yrow + s) = make_uint2(lo, hi);
        }
    }
}

// ------------------------------------------------------------------ step 2: the sum of shifted rows
struct RowsArgs {
    const void *y;                    // [nslots][nyrows][ystride] pre-summed rows
    void *out;
    const int4 *rowdesc;              // [nblk][nslab][CS]: (y row or -1, first staged sample - tile_t0, samples to copy, 0)
    const uint32_t *ent;              // [nblk][nslab][warp][Q][D] byte offset of the (DM, group) window inside a stage (uint16: | odd)
    const int32_t *sigma;             // [DB] output time shear per DM of a block
    int beam0, nslots, nyrows, ndms;
    int nblk, ntile_t, nslab, Q, ngroups, CS, pitch, stages, slabs_per_part;
    int stride;                       // outputs a tile owns per DM (its time step)
    long long ntiles, nsamps, nsamps_out, ystride;
};

// F32_: 32-bit rows, one sample per word (INT_ = false: float adds, MDSM_F32; INT_ = true: integer adds, MDSM_U16);
// !F32_: 16-bit rows packed two per word (MDSM_U8, MDSM_U4).
template <int D_, int T_, int NW_, bool F32_, bool INT_ = false> struct RowsTraits {
    static constexpr int D = D_, T = T_, NW = NW_;
    static constexpr bool kF32 = F32_;
    using Acc = typename std::conditional<INT_, uint32_t, float>::type;
    static constexpr int kSpan = F32_ ? 32 * T_ : 64 * T_;          // samples a warp's accumulators cover per DM
    using Y = typename std::conditional<F32_, float, uint16_t>::type;
};

template <typename Tr>
__global__ void __launch_bounds__((Tr::NW + 1) * 32, 1) dedisperse_rows_kernel(const RowsArgs a)
{
    using Y = typename Tr::Y;
    constexpr int D = Tr::D, T = Tr::T, NW = Tr::NW, DB = D * NW;
    extern __shared__ __align__(128) unsigned char smem[];
    const int stages = a.stages;
    const uint32_t row_bytes = (uint32_t)a.pitch * sizeof(Y);
    const uint32_t ent_bytes = (uint32_t)(DB * a.Q) * 4u;
    const uint32_t stage_bytes = (a.CS * row_bytes + ent_bytes + 127u) & ~127u;     // rows, then the entry slice
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + (size_t)stages * stage_bytes);
    uint64_t *empty = full + stages;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    // Rows that stick out of [0, ystride) are only partly written by the bulk copies.  What they leave behind feeds
    // outputs outside [0, nsamps_out) only, but a stale 16-bit lane must never carry into its valid neighbour: with
    // the stages zeroed once, every staged value is zero or a real group sum.
    for (uint32_t i = threadIdx.x; i < stages * stage_bytes / 16; i += blockDim.x) reinterpret_cast<uint4 *>(smem)[i] = make_uint4(0, 0, 0, 0);
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    if (threadIdx.x == 0) {
        for (int s = 0; s < stages; ++s) {
            mbar_init(&full[s], 32);
            mbar_init(&empty[s], NW);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp == NW) {
        // ===== producer: lane r copies rows r and r + 32 of every slab, lane 0 also the slab's slice of the entry table =====
        int st = 0;
        uint32_t ph = 1;             // parity of the empty-barrier phase to wait for (first lap: no wait)
        bool first_lap = true;
        const uint32_t smem0 = smem_u32(smem);
        const int4 none = make_int4(-1, 0, 0, 0);
        for (long long tile = blockIdx.x; tile < a.ntiles; tile += gridDim.x) {
            const int blk = (int)(tile % a.nblk);
            const long long rest = tile / a.nblk;
            const int tt = (int)(rest % a.ntile_t), bb = (int)(rest / a.ntile_t);
            const long long tile_t0 = (long long)tt * a.stride;
            const Y *ybeam = reinterpret_cast<const Y *>(a.y) + (size_t)((a.beam0 + bb) % a.nslots) * a.nyrows * (size_t)a.ystride;
            const int4 *rd = a.rowdesc + (size_t)blk * a.nslab * a.CS;
            const uint32_t *et = a.ent + (size_t)blk * a.nslab * (DB * a.Q);
            int4 desc0 = lane < a.CS ? rd[lane] : none, desc1 = lane + 32 < a.CS ? rd[lane + 32] : none;
            for (int slab = 0; slab < a.nslab; ++slab) {
                const int4 cur[2] = {desc0, desc1};
                if (slab + 1 < a.nslab) {                                  // next slab's rows, before the wait
                    if (lane < a.CS) desc0 = rd[(size_t)(slab + 1) * a.CS + lane];
                    if (lane + 32 < a.CS) desc1 = rd[(size_t)(slab + 1) * a.CS + lane + 32];
                }
                if (!first_lap) mbar_wait_sleep(&empty[st], ph);
                const uint32_t sbase = smem0 + st * stage_bytes;
                uint32_t bytes[2] = {0, 0};
                long long lo[2] = {0, 0}, g0[2] = {0, 0};
#pragma unroll
                for (int k = 0; k < 2; ++k)
                    if (cur[k].x >= 0) {
                        g0[k] = tile_t0 + cur[k].y;
                        lo[k] = g0[k] < 0 ? 0 : g0[k];
                        long long hi = g0[k] + cur[k].z;
                        if (hi > a.ystride) hi = a.ystride;
                        if (hi > lo[k]) bytes[k] = (uint32_t)((hi - lo[k]) * sizeof(Y));
                    }
                mbar_arrive_expect_tx(&full[st], bytes[0] + bytes[1] + (lane == 0 ? ent_bytes : 0u));
#pragma unroll
                for (int k = 0; k < 2; ++k)
                    if (bytes[k])
                        bulk_g2s(sbase + (lane + 32 * k) * row_bytes + (uint32_t)((lo[k] - g0[k]) * sizeof(Y)),
                                 ybeam + (size_t)cur[k].x * a.ystride + lo[k], bytes[k], &full[st]);
                if (lane == 0) bulk_g2s(sbase + a.CS * row_bytes, et + (size_t)slab * (DB * a.Q), ent_bytes, &full[st]);
                if (++st == stages) { st = 0; ph ^= 1; first_lap = false; }
            }
        }
        return;
    }

    // ===== consumer warps =====
    const int Q = a.Q;
    int st = 0;
    uint32_t ph = 0;
    for (long long tile = blockIdx.x; tile < a.ntiles; tile += gridDim.x) {
        const int blk = (int)(tile % a.nblk);
        const long long rest = tile / a.nblk;
        const int tt = (int)(rest % a.ntile_t), bb = (int)(rest / a.ntile_t);
        const long long tile_t0 = (long long)tt * a.stride;
        const int b = a.beam0 + bb;
        if constexpr (Tr::kF32) {
            using Acc = typename Tr::Acc;
            Acc acc[D][T];
#pragma unroll
            for (int j = 0; j < D; ++j)
#pragma unroll
                for (int i = 0; i < T; ++i) acc[j][i] = (Acc)0;
#pragma unroll 1
            for (int slab = 0; slab < a.nslab; ++slab) {
                const int nq = min(Q, a.ngroups - slab * Q);
                mbar_wait(&full[st], ph);
                const unsigned char *sbase = smem + (size_t)st * stage_bytes;
                const uint32_t *ents = reinterpret_cast<const uint32_t *>(sbase + a.CS * row_bytes) + warp * D * Q;
#pragma unroll 1
                for (int q = 0; q < nq; ++q) {
                    uint32_t e[D];
                    if constexpr (D == 4) {                                             // four consecutive words: one 128-bit broadcast load
                        const uint4 ev = *reinterpret_cast<const uint4 *>(ents + q * 4);
                        e[0] = ev.x; e[1] = ev.y; e[2] = ev.z; e[3] = ev.w;
                    } else {
#pragma unroll
                        for (int j = 0; j < D; ++j) e[j] = ents[q * D + j];
                    }
#pragma unroll
                    for (int j = 0; j < D; ++j) {
                        const Acc *w = reinterpret_cast<const Acc *>(sbase + e[j]) + lane;
                        Acc v[T];
#pragma unroll
                        for (int i = 0; i < T; ++i) v[i] = w[32 * i];
#pragma unroll
                        for (int i = 0; i < T; ++i) acc[j][i] += v[i];
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(&empty[st]);
                if (++st == stages) { st = 0; ph ^= 1; }
            }
#pragma unroll
            for (int j = 0; j < D; ++j) {
                const int dl = warp * D + j, d = blk * DB + dl;
                if (d >= a.ndms) continue;
                const int sg = a.sigma[dl];
                Acc *orow = reinterpret_cast<Acc *>(a.out) + ((size_t)b * a.ndms + d) * (size_t)a.nsamps;
#pragma unroll
                for (int i = 0; i < T; ++i) {
                    const long long t = tile_t0 - sg + lane + 32 * i;
                    if (t >= 0 && t < a.nsamps_out) orow[t] = acc[j][i];
                }
            }
        } else {
            uint32_t accE[D][T], accO[D][T];
#pragma unroll 1
            for (int s0 = 0; s0 < a.nslab; s0 += a.slabs_per_part) {
#pragma unroll
                for (int j = 0; j < D; ++j)
#pragma unroll
                    for (int i = 0; i < T; ++i) { accE[j][i] = 0; accO[j][i] = 0; }
                const int s1 = min(a.nslab, s0 + a.slabs_per_part);
#pragma unroll 1
                for (int slab = s0; slab < s1; ++slab) {
                    const int nq = min(Q, a.ngroups - slab * Q);
                    mbar_wait(&full[st], ph);
                    const unsigned char *sbase = smem + (size_t)st * stage_bytes;
                    const uint32_t *ents = reinterpret_cast<const uint32_t *>(sbase + a.CS * row_bytes) + warp * D * Q;
#pragma unroll 1
                    for (int q = 0; q < nq; ++q) {
                        uint32_t e[D];
                        if constexpr (D == 4) {
                            const uint4 ev = *reinterpret_cast<const uint4 *>(ents + q * 4);
                            e[0] = ev.x; e[1] = ev.y; e[2] = ev.z; e[3] = ev.w;
                        } else {
#pragma unroll
                            for (int j = 0; j < D; ++j) e[j] = ents[q * D + j];
                        }               // D consecutive words: one broadcast load
#pragma unroll
                        for (int j = 0; j < D; ++j) {
                            const uint32_t *w = reinterpret_cast<const uint32_t *>(sbase + (e[j] & ~3u)) + lane;
                            uint32_t v[T];
#pragma unroll
                            for (int i = 0; i < T; ++i) v[i] = w[32 * i];
                            if (e[j] & 1u) {
#pragma unroll
                                for (int i = 0; i < T; ++i) accO[j][i] += v[i];
                            } else {
#pragma unroll
                                for (int i = 0; i < T; ++i) accE[j][i] += v[i];
                            }
                        }
                    }
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&empty[st]);
                    if (++st == stages) { st = 0; ph ^= 1; }
                }
                // ----- flush of the part: out(2k) = E_k.lo + O_k.hi, out(2k+1) = E_k.hi + O_{k+1}.lo, word k = lane + 32 i -----
#pragma unroll
                for (int j = 0; j < D; ++j) {
                    const int dl = warp * D + j, d = blk * DB + dl;
                    const long long ts = tile_t0 - a.sigma[dl] + 2 * lane;
                    uint32_t *orow = reinterpret_cast<uint32_t *>(a.out) + ((size_t)b * a.ndms + (d < a.ndms ? d : 0)) * (size_t)a.nsamps;
                    uint32_t v0[T], v1[T];
                    bool ok0[T], ok1[T];
#pragma unroll
                    for (int i = 0; i < T; ++i) {
                        const uint32_t up = __shfl_sync(0xffffffffu, accO[j][i], (lane + 1) & 31);
                        const uint32_t wrap = __shfl_sync(0xffffffffu, accO[j][i + 1 < T ? i + 1 : i], 0);
                        const uint32_t onext = lane == 31 ? wrap : up;
                        v0[i] = (accE[j][i] & 0xffffu) + (accO[j][i] >> 16);
                        v1[i] = (accE[j][i] >> 16) + (onext & 0xffffu);
                        const int k2 = 2 * (lane + 32 * i);
                        const long long t = ts + 64 * i;
                        ok0[i] = d < a.ndms && k2 < a.stride && t >= 0 && t < a.nsamps_out;
                        ok1[i] = d < a.ndms && k2 + 1 < a.stride && t + 1 >= 0 && t + 1 < a.nsamps_out;
                    }
                    if (s0 != 0) {
                        // later parts add to what part 0 stored: this thread's own elements (still in L2); all the loads
                        // are issued before the first store so that their latencies overlap
                        uint32_t o0[T], o1[T];
#pragma unroll
                        for (int i = 0; i < T; ++i) {
                            o0[i] = ok0[i] ? __ldcg(orow + ts + 64 * i) : 0u;
                            o1[i] = ok1[i] ? __ldcg(orow + ts + 64 * i + 1) : 0u;
                        }
#pragma unroll
                        for (int i = 0; i < T; ++i) { v0[i] += o0[i]; v1[i] += o1[i]; }
                    }
#pragma unroll
                    for (int i = 0; i < T; ++i) {
                        if (ok0[i]) orow[ts + 64 * i] = v0[i];
                        if (ok1[i]) orow[ts + 64 * i + 1] = v1[i];
                    }
                }
            }
        }
    }
}

// ------------------------------------------------------------------ step 2, TMEM variant (fp32)
// The rows kernel above is bound by the shared-memory pipe: one 32-bit operand word per add, 32 words per clock and SM.
// Tensor memory (TMEM, 128 lanes x 512 columns x 32 bit per SM) has its own read path into the register file
// (tcgen05.ld), measured at ~3x that rate with the adds in the loop, and -- unlike registers -- its COLUMN address is
// a run-time value.  So the operand window moves there:
//   * TMEM lane l of a quadrant holds the samples  s0 + P l + [0, 16 + S)  of a staged y row in consecutive columns
//     (P = 15 outputs per lane and DM, S = spread of the window starts of the DMs that use the row);
//   * a consumer thread (lane l) owns the P consecutive outputs  tile_t0 - sigma_d + P l + [0, P)  of each of its D DMs
//     and fetches, per (DM, group), 16 consecutive columns at the DM's own column offset: one tcgen05.ld.32x32b.x16 per
//     15 adds, no alignment cases, no shared-memory traffic;
//   * the rows get into TMEM through the consumer warps themselves: TMEM lanes are only reachable from the warps w with
//     w % 4 == quadrant, so the 4 warps of a quadrant share the copy of the rows their 16 DMs use, 16 columns at a time
//     (conflict-free 32-bit shared-memory loads because P is odd, then tcgen05.st).  A staged word serves every DM of
//     the quadrant that uses the row, so the shared-memory pipe carries ~0.5 words per add instead of 1.
// Warps: 16 consumers (quadrant = w & 3, D DMs each) and 1 TMA producer (w = 16; its warpgroup hands registers to the
// consumers with setmaxnreg).  Rings: shared-memory stages (producer -> consumers' staging half), two TMEM buffers of 256
// columns per quadrant (staging half -> adding half of the same four warps, one slab ahead).
constexpr int kTmWarps = 20;          // 16 consumers + the producer's warpgroup (3 of its warps idle)
constexpr int kTmProducer = 16;
constexpr int kTmCols = 256;          // TMEM columns per buffer (two buffers)
constexpr int kTmQMax = 4;            // most groups per slab
constexpr int kTmCQMax = 32;          // most 16-column chunks per quadrant and slab
constexpr int kTmEnt = 20;            // words of a warp's entry copy (D * kTmQMax entries + the group count, padded)

struct TmemArgs {
    const float *y;
    float *out;
    const int4 *rowdesc;              // [nblk][nslab_max][CS]: (y row or -1, first staged sample - tile_t0, samples, 0)
    const uint32_t *tab;              // [nblk][nslab_max][tabw]
    const int32_t *nslab;             // [nblk]
    const int32_t *sigma;             // [DB]
    int beam0, nslots, nyrows, ndms;
    int nblk, ntile_t, nslab_max, CS, pitch, stages, tabw, span;
    long long ntiles, nsamps, nsamps_out, ystride;
};

__device__ __forceinline__ void tm_ld16(uint32_t taddr, uint32_t (&r)[16])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
                   "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
                 : "r"(taddr));
}
__device__ __forceinline__ void tm_st8(uint32_t taddr, const uint32_t (&r)[8])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"r"(taddr), "r"(r[0]), "r"(r[1]),
                 "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7])
                 : "memory");
}
__device__ __forceinline__ void tm_st16(uint32_t taddr, const uint32_t (&r)[16])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};" ::"r"(taddr),
                 "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]), "r"(r[10]),
                 "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15])
                 : "memory");
}
__device__ __forceinline__ void tm_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tm_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tm_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tm_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

// walks the slabs of the tiles a CTA owns, in order
struct TmSlabIter {
    long long tile;
    int blk, nslab, slab;
    __device__ __forceinline__ void init(const TmemArgs &a)
    {
        tile = blockIdx.x;
        slab = 0;
        load(a);
    }
    __device__ __forceinline__ void load(const TmemArgs &a)
    {
        if (tile < a.ntiles) { blk = (int)(tile % a.nblk); nslab = a.nslab[blk]; }
    }
    __device__ __forceinline__ bool valid(const TmemArgs &a) const { return tile < a.ntiles; }
    __device__ __forceinline__ void advance(const TmemArgs &a)
    {
        if (++slab == nslab) { slab = 0; tile += gridDim.x; load(a); }
    }
};

template <int D, int P>
__global__ void __launch_bounds__(kTmWarps * 32, 1) dedisperse_tmem_kernel(const TmemArgs a)
{
    static_assert(P % 2 == 1 && P <= 16, "P must be odd (conflict-free staging) and fit one x16 load");
    static_assert(D * kTmQMax + 1 <= kTmEnt, "entry copy too small");
    constexpr int DQ = 4 * D, DB = 16 * D;
    extern __shared__ __align__(128) unsigned char smem[];
    const int stages = a.stages;
    const uint32_t row_bytes = (uint32_t)a.pitch * 4u;
    const uint32_t tab_bytes = (uint32_t)a.tabw * 4u;
    const uint32_t stage_bytes = (a.CS * row_bytes + tab_bytes + 127u) & ~127u;
    uint32_t *tent = reinterpret_cast<uint32_t *>(smem + (size_t)stages * stage_bytes);       // [2][16][kTmEnt]
    uint64_t *full = reinterpret_cast<uint64_t *>(tent + 2 * 16 * kTmEnt);
    uint64_t *empty = full + stages;
    uint64_t *tfull = empty + stages;          // [2][4]
    uint64_t *tempty = tfull + 8;              // [2][4]
    uint32_t *tbase_slot = reinterpret_cast<uint32_t *>(tempty + 8);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    for (uint32_t i = threadIdx.x; i < stages * stage_bytes / 16; i += blockDim.x) reinterpret_cast<uint4 *>(smem)[i] = make_uint4(0, 0, 0, 0);
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    if (threadIdx.x == 0) {
        for (int s = 0; s < stages; ++s) {
            mbar_init(&full[s], 32);
            mbar_init(&empty[s], 16);
        }
        for (int s = 0; s < 8; ++s) {
            mbar_init(&tfull[s], 4);
            mbar_init(&tempty[s], 4);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == kTmProducer) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(tbase_slot)));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    tm_fence_before();
    __syncthreads();
    tm_fence_after();
    const uint32_t tbase = *tbase_slot;
    if (warp >= kTmProducer) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 40;");
      if (warp == kTmProducer) {
        // ===== TMA producer: lane r copies row r of every slab, lane 0 also the slab's table slice =====
        int st = 0;
        uint32_t ph = 1;
        bool first_lap = true;
        const uint32_t smem0 = smem_u32(smem);
        for (long long tile = blockIdx.x; tile < a.ntiles; tile += gridDim.x) {
            const int blk = (int)(tile % a.nblk);
            const long long rest = tile / a.nblk;
            const int tt = (int)(rest % a.ntile_t), bb = (int)(rest / a.ntile_t);
            const long long tile_t0 = (long long)tt * a.span;
            const float *ybeam = a.y + (size_t)((a.beam0 + bb) % a.nslots) * a.nyrows * (size_t)a.ystride;
            const int4 *rd = a.rowdesc + (size_t)blk * a.nslab_max * a.CS;
            const uint32_t *tb = a.tab + (size_t)blk * a.nslab_max * a.tabw;
            const int nslab = a.nslab[blk];
            int4 desc = lane < a.CS ? rd[lane] : make_int4(-1, 0, 0, 0);
            for (int slab = 0; slab < nslab; ++slab) {
                const int4 cur = desc;
                if (slab + 1 < nslab && lane < a.CS) desc = rd[(size_t)(slab + 1) * a.CS + lane];
                if (!first_lap) mbar_wait_sleep(&empty[st], ph);
                const uint32_t sbase = smem0 + st * stage_bytes;
                uint32_t bytes = 0;
                long long lo = 0, g0 = 0;
                if (cur.x >= 0) {
                    g0 = tile_t0 + cur.y;
                    lo = g0 < 0 ? 0 : g0;
                    long long hi = g0 + cur.z;
                    if (hi > a.ystride) hi = a.ystride;
                    if (hi > lo) bytes = (uint32_t)((hi - lo) * 4);
                }
                mbar_arrive_expect_tx(&full[st], bytes + (lane == 0 ? tab_bytes : 0u));
                if (bytes) bulk_g2s(sbase + lane * row_bytes + (uint32_t)((lo - g0) * 4), ybeam + (size_t)cur.x * a.ystride + lo, bytes, &full[st]);
                if (lane == 0) bulk_g2s(sbase + a.CS * row_bytes, tb + (size_t)slab * a.tabw, tab_bytes, &full[st]);
                if (++st == stages) { st = 0; ph ^= 1; first_lap = false; }
            }
        }
      }
    } else {
        asm volatile("setmaxnreg.inc.sync.aligned.u32 104;");
        // ===== consumers: warp (q, sub) owns the DMs q DQ + sub D + j of the block; the four warps of a quadrant stage the
        // quadrant's rows of slab n + 1 into TMEM buffer (n + 1) & 1, then add slab n out of buffer n & 1 =====
        const int q = warp & 3, sub = warp >> 2;
        const uint32_t tq = tbase + ((uint32_t)(q * 32) << 16);
        uint32_t *my_ent = tent + warp * kTmEnt;                 // + buffer * 16 * kTmEnt
        TmSlabIter si, ci;
        si.init(a);
        ci.init(a);
        uint32_t nstaged = 0, nadded = 0;                        // slabs staged / added so far by this warp
        int sst = 0;                                             // shared-memory stage of the next slab to stage
        uint32_t sph = 0;

        auto stage_one = [&]() {
            const int buf = nstaged & 1;
            mbar_wait(&full[sst], sph);
            if (nstaged >= 2) {                                  // the buffer's previous slab must have been added by all four warps
                while (!mbar_try_wait(&tempty[buf * 4 + q], ((nstaged >> 1) - 1) & 1)) {}
            }
            tm_fence_after();
            const unsigned char *sbase = smem + (size_t)sst * stage_bytes;
            const uint32_t *tab = reinterpret_cast<const uint32_t *>(sbase + a.CS * row_bytes);
            const int nch = (int)tab[q];
            const float *rows = reinterpret_cast<const float *>(sbase) + P * lane;
            const uint32_t tbuf = tq + buf * kTmCols;
#pragma unroll 1
            for (int j = sub; j < nch; j += 4) {
                const uint32_t soff = tab[8 + (q * kTmCQMax + j) * 2], w1 = tab[8 + (q * kTmCQMax + j) * 2 + 1];
                const float *src = rows + soff;
                const uint32_t tcol = tbuf + (w1 & 0xffffu);
                if (w1 >> 16) {                                  // 16 columns
                    uint32_t v[16];
#pragma unroll
                    for (int i = 0; i < 16; ++i) v[i] = __float_as_uint(src[i]);
                    tm_st16(tcol, v);
                } else {
                    uint32_t v[8];
#pragma unroll
                    for (int i = 0; i < 8; ++i) v[i] = __float_as_uint(src[i]);
                    tm_st8(tcol, v);
                }
            }
            // this warp's entries (TMEM column per (DM, group)) and the number of groups of the slab
            const uint32_t *ent = tab + 8 + 4 * kTmCQMax * 2 + (q * DQ + sub * D) * kTmQMax;
            uint32_t *te = my_ent + buf * 16 * kTmEnt;
            if (lane < D * kTmQMax) te[lane] = ent[lane];
            if (lane == 31) te[D * kTmQMax] = tab[4];
            tm_wait_st();
            tm_fence_before();
            __syncwarp();
            if (lane == 0) {
                mbar_arrive(&tfull[buf * 4 + q]);
                mbar_arrive(&empty[sst]);
            }
            if (++sst == stages) { sst = 0; sph ^= 1; }
            ++nstaged;
        };

        if (si.valid(a)) { stage_one(); si.advance(a); }
        while (ci.valid(a)) {
            const long long rest = ci.tile / a.nblk;
            const int tt = (int)(rest % a.ntile_t), bb = (int)(rest / a.ntile_t);
            const long long tile_t0 = (long long)tt * a.span;
            const int blk = ci.blk, nslab = ci.nslab;
            float acc[D][P];
#pragma unroll
            for (int j = 0; j < D; ++j)
#pragma unroll
                for (int i = 0; i < P; ++i) acc[j][i] = 0.0f;
#pragma unroll 1
            for (int slab = 0; slab < nslab; ++slab) {
                if (si.valid(a)) { stage_one(); si.advance(a); }
                const int buf = nadded & 1;
                while (!mbar_try_wait(&tfull[buf * 4 + q], (nadded >> 1) & 1)) {}
                tm_fence_after();
                const uint32_t *te = my_ent + buf * 16 * kTmEnt;
                const int nq = (int)te[D * kTmQMax];
                const uint32_t tbuf = tq + buf * kTmCols;
#pragma unroll 1
                for (int g = 0; g < nq; ++g) {
                    uint32_t e[D];
#pragma unroll
                    for (int j = 0; j < D; ++j) e[j] = te[j * kTmQMax + g];
#pragma unroll
                    for (int j = 0; j < D; ++j) {
                        uint32_t v[16];
                        tm_ld16(tbuf + e[j], v);
                        tm_wait_ld();
#pragma unroll
                        for (int i = 0; i < P; ++i) acc[j][i] += __uint_as_float(v[i]);
                    }
                }
                tm_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(&tempty[buf * 4 + q]);
                ++nadded;
                ci.advance(a);
            }
            const int b = a.beam0 + bb;
#pragma unroll
            for (int j = 0; j < D; ++j) {
                const int dl = q * DQ + sub * D + j, d = blk * DB + dl;
                if (d >= a.ndms) continue;
                const long long ts0 = tile_t0 - a.sigma[dl] + P * lane;
                float *orow = a.out + ((size_t)b * a.ndms + d) * (size_t)a.nsamps;
#pragma unroll
                for (int i = 0; i < P; ++i) {
                    const long long t = ts0 + i;
                    if (t >= 0 && t < a.nsamps_out) orow[t] = acc[j][i];
                }
            }
        }
    }
    tm_fence_before();
    __syncthreads();
    if (warp == kTmProducer) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tbase));
}


// ------------------------------------------------------------------ host side: the plan-time tables
struct RowsGeom { int D, T, NW; };
constexpr RowsGeom kGeomRowsF32 = {4, 16, 16};      // 64 DMs x 512 samples per tile
constexpr RowsGeom kGeomRowsU16 = {4, 8, 16};       // 64 DMs x 512 samples (504 owned) per tile
constexpr int kPartChansU8 = 256;                   // 256 * 255 < 2^16: the most uint8 channels a 16-bit lane can take
constexpr int kPartChansU4 = 4096;                  // 4096 * 15 < 2^16: the same for 4-bit samples
constexpr size_t kSmemBudget = 227 * 1024;

static inline long long floor_to(long long v, int a) { return v >= 0 ? (v / a) * a : -(((-v) + a - 1) / a) * a; }
static inline long long ceil_to(long long v, int a) { return -floor_to(-v, a); }

template <typename V> static bool upload(V **dptr, const std::vector<V> &h)
{
    if (cudaMalloc((void **)dptr, std::max<size_t>(h.size(), 1) * sizeof(V)) != cudaSuccess) return false;
    return h.empty() || cudaMemcpy(*dptr, h.data(), h.size() * sizeof(V), cudaMemcpyHostToDevice) == cudaSuccess;
}

// y rows of a group size: every pattern of relative delays a group takes over the DM grid
struct GroupRows {
    int G = 0, ngroups = 0, nyrows = 0, dmax = 0, maxpat = 0;  // maxpat: most rows of one group
    std::vector<int32_t> yrow_of;          // [ndms][ngroups]
    std::vector<int32_t> group_row0;       // [ngroups + 1]
    std::vector<int16_t> ydelta;           // [nyrows][kGMax]
};

static bool enumerate_group_rows(const mdsm_plan *p, int G, GroupRows &gr)
{
    gr.G = G;
    gr.ngroups = (p->nchans + G - 1) / G;
    gr.yrow_of.assign((size_t)p->ndms * gr.ngroups, 0);
    gr.group_row0.assign(gr.ngroups + 1, 0);
    gr.ydelta.clear();
    gr.dmax = 0;
    int nrows = 0;
    for (int g = 0; g < gr.ngroups; ++g) {
        gr.group_row0[g] = nrows;
        std::map<std::array<int16_t, kGMax>, int> seen;
        const int c0 = g * G;
        std::array<int16_t, kGMax> last{};
        int last_row = -1;
        for (int d = 0; d < p->ndms; ++d) {
            const int32_t *row = p->h_delay.data() + (size_t)d * p->nchans;
            std::array<int16_t, kGMax> pat{};
            for (int i = 1; i < G && c0 + i < p->nchans; ++i) {
                const long long de = (long long)row[c0 + i] - row[c0];
                if (de < 0 || de > 4000) return false;          // not a dispersion sweep this scheme is meant for
                pat[i] = (int16_t)de;
                gr.dmax = std::max(gr.dmax, (int)de);
            }
            if (d > 0 && pat == last) {                         // neighbouring DMs mostly share the pattern
                gr.yrow_of[(size_t)d * gr.ngroups + g] = last_row;
                continue;
            }
            auto it = seen.find(pat);
            if (it == seen.end()) {
                it = seen.emplace(pat, nrows++).first;
                gr.ydelta.insert(gr.ydelta.end(), pat.begin(), pat.end());
            }
            gr.yrow_of[(size_t)d * gr.ngroups + g] = it->second;
            last = pat;
            last_row = it->second;
        }
    }
    gr.group_row0[gr.ngroups] = nrows;
    gr.nyrows = nrows;
    gr.maxpat = 0;
    for (int g = 0; g < gr.ngroups; ++g) gr.maxpat = std::max(gr.maxpat, gr.group_row0[g + 1] - gr.group_row0[g]);
    return true;
}

struct RowsHost {
    std::vector<int4> rowdesc;
    std::vector<uint32_t> ent;
    std::vector<int32_t> sigma;
};

// Builds the per-block staging lists and entry tables for one dtype, group size and geometry.
static bool build_rows_tables(const mdsm_plan *p, bool f32, int part_chans, const GroupRows &gr, const RowsGeom &g, RowsTables &rt, RowsHost &h)
{
    const int al = f32 ? 4 : 8, esize = f32 ? 4 : 2;
    const int DB = g.D * g.NW;
    const int span = f32 ? 32 * g.T : 64 * g.T;
    const int stride = f32 ? span : span - 8;
    const int nblk = (p->ndms + DB - 1) / DB;
    const int ng = gr.ngroups, G = gr.G;
    // un-rounded delay increment per DM step at the band edge: the slope the shear splits in half
    const double f_lo = p->f_top + (p->nchans - 1) * p->foff;
    const double smax = 4.148808e3 * p->dm_step * (1.0 / (f_lo * f_lo) - 1.0 / (p->f_top * p->f_top)) / p->tsamp;
    h.sigma.resize(DB);
    for (int dl = 0; dl < DB; ++dl) h.sigma[dl] = (int32_t)llround(0.5 * smax * dl);
    auto dly = [&](int d, int c) { return (long long)p->h_delay[(size_t)d * p->nchans + c]; };

    // per block and group: the distinct y rows its DMs use, with the range of window starts
    struct Use { int yrow; long long emin, emax; };
    std::vector<std::vector<Use>> uses((size_t)nblk * ng);
    long long need_max = 0;
    for (int blk = 0; blk < nblk; ++blk)
        for (int gi = 0; gi < ng; ++gi) {
            auto &u = uses[(size_t)blk * ng + gi];
            for (int dl = 0; dl < DB; ++dl) {
                const int d = blk * DB + dl;
                if (d >= p->ndms) break;
                const int yr = gr.yrow_of[(size_t)d * ng + gi];
                const long long e = dly(d, gi * G) - h.sigma[dl];
                auto it = std::find_if(u.begin(), u.end(), [&](const Use &x) { return x.yrow == yr; });
                if (it == u.end()) u.push_back({yr, e, e});
                else { it->emin = std::min(it->emin, e); it->emax = std::max(it->emax, e); }
            }
            for (const Use &x : u) need_max = std::max(need_max, x.emax - floor_to(x.emin, al) + span);
        }
    const int pitch = (int)ceil_to(need_max, al);
    // groups per slab: as many as keep a slab within 64 rows (two per producer lane) and three stages in shared memory
    const int part_groups_max = f32 ? ng : std::max(1, part_chans / G);
    int Q = 0, CS = 0;
    for (int q : {4, 3, 2, 1}) {
        if (!f32 && part_groups_max % q) continue;
        if ((DB * q) % 4) continue;
        int cs = 0;
        for (int blk = 0; blk < nblk; ++blk)
            for (int s0 = 0; s0 < ng; s0 += q) {
                int n = 0;
                for (int gi = s0; gi < std::min(ng, s0 + q); ++gi) n += (int)uses[(size_t)blk * ng + gi].size();
                cs = std::max(cs, n);
            }
        const size_t stage = (((size_t)cs * pitch * esize + (size_t)DB * q * 4) + 127) & ~(size_t)127;
        if (cs <= 64 && 2 * stage + 256 <= kSmemBudget) { Q = q; CS = cs; break; }
    }
    if (!Q) return false;
    const int nslab = (ng + Q - 1) / Q;
    h.rowdesc.assign((size_t)nblk * nslab * CS, make_int4(-1, 0, 0, 0));
    h.ent.assign((size_t)nblk * nslab * DB * Q, 0u);
    for (int blk = 0; blk < nblk; ++blk)
        for (int slab = 0; slab < nslab; ++slab) {
            int r = 0;
            for (int q = 0; q < Q; ++q) {
                const int gi = slab * Q + q;
                if (gi >= ng) break;
                const auto &u = uses[(size_t)blk * ng + gi];
                for (size_t k = 0; k < u.size(); ++k) {
                    const long long rs = floor_to(u[k].emin, al);
                    const long long len = ceil_to(u[k].emax - rs + span, al);
                    h.rowdesc[((size_t)blk * nslab + slab) * CS + r + k] = make_int4(u[k].yrow, (int)rs, (int)len, 0);
                }
                for (int dl = 0; dl < DB; ++dl) {
                    const int d = std::min(blk * DB + dl, p->ndms - 1);
                    const int dle = d - blk * DB;                           // a DM past the grid repeats the last one (never stored)
                    const int yr = gr.yrow_of[(size_t)d * ng + gi];
                    size_t k = 0;
                    while (u[k].yrow != yr) ++k;
                    const long long o = dly(d, gi * G) - h.sigma[dle] - floor_to(u[k].emin, al);
                    uint32_t e;
                    if (f32) e = (uint32_t)(((long long)(r + k) * pitch + o) * 4);
                    else e = (uint32_t)(((long long)(r + k) * pitch + (o & ~1LL)) * 2) | (uint32_t)(o & 1);
                    h.ent[((size_t)blk * nslab + slab) * DB * Q + ((size_t)(dl / g.D) * Q + q) * g.D + dl % g.D] = e;   // [warp][group][DM of the warp]
                }
                r += (int)u.size();
            }
        }
    rt.G = G; rt.D = g.D; rt.T = g.T; rt.NW = g.NW; rt.DB = DB; rt.span = span; rt.stride = stride;
    rt.Q = Q; rt.CS = CS; rt.pitch = pitch; rt.nslab = nslab; rt.nblk = nblk; rt.ngroups = ng; rt.nyrows = gr.nyrows;
    rt.dmax = gr.dmax;
    rt.maxpat = gr.maxpat;
    rt.slabs_per_part = f32 ? nslab : part_groups_max / Q;
    rt.ystride = ceil_to(p->nsamps, al);
    rt.sigma_max = *std::max_element(h.sigma.begin(), h.sigma.end());
    const size_t stage = (((size_t)CS * pitch * esize + (size_t)DB * Q * 4) + 127) & ~(size_t)127;
    rt.stages = (int)std::min<size_t>(8, (kSmemBudget - 256) / stage);
    rt.smem_bytes = (size_t)rt.stages * stage + 2 * rt.stages * sizeof(uint64_t);
    long long rows_staged = 0;
    for (const auto &u : uses) rows_staged += (long long)u.size();
    rt.rows_per_block = (double)rows_staged / nblk;
    return true;
}

// ---- tables of the TMEM variant (fp32): variable slabs of <= kTmQMax groups, packed so that every quadrant's rows fit a
// TMEM stage of kTmCols columns and the block's rows fit the shared-memory stage.
struct TmemGeom { int D, P; };
constexpr TmemGeom kGeomTmem = {4, 15};            // 64 DMs x 480 samples per tile

struct TmemHost {
    std::vector<int4> rowdesc;
    std::vector<uint32_t> tab;
    std::vector<int32_t> nslab, sigma;
};

static bool build_tmem_tables(const mdsm_plan *p, const GroupRows &gr, TmemTables &tt, TmemHost &h)
{
    const int D = kGeomTmem.D, P = kGeomTmem.P, DQ = 4 * D, DB = 16 * D, span = 32 * P, al = 4;
    const int nblk = (p->ndms + DB - 1) / DB, ng = gr.ngroups, G = gr.G;
    const double f_lo = p->f_top + (p->nchans - 1) * p->foff;
    const double smax = 4.148808e3 * p->dm_step * (1.0 / (f_lo * f_lo) - 1.0 / (p->f_top * p->f_top)) / p->tsamp;
    h.sigma.resize(DB);
    for (int dl = 0; dl < DB; ++dl) h.sigma[dl] = (int32_t)llround(0.5 * smax * dl);
    auto dly = [&](int d, int c) { return (long long)p->h_delay[(size_t)d * p->nchans + c]; };
    struct Use { int yrow; long long emin, emax; };
    struct GroupUse { std::vector<Use> blk; std::vector<Use> quad[4]; int cols[4], chunks[4]; };
    auto add_use = [](std::vector<Use> &u, int yr, long long e) {
        auto it = std::find_if(u.begin(), u.end(), [&](const Use &x) { return x.yrow == yr; });
        if (it == u.end()) u.push_back({yr, e, e});
        else { it->emin = std::min(it->emin, e); it->emax = std::max(it->emax, e); }
    };
    const int tabw = 8 + 4 * kTmCQMax * 2 + DB * kTmQMax;
    std::vector<std::vector<GroupUse>> gu(nblk, std::vector<GroupUse>(ng));
    long long need_max = 0;
    for (int blk = 0; blk < nblk; ++blk)
        for (int gi = 0; gi < ng; ++gi) {
            GroupUse &u = gu[blk][gi];
            for (int dl = 0; dl < DB; ++dl) {
                const int d = std::min(blk * DB + dl, p->ndms - 1), dle = d - blk * DB;     // DMs past the grid repeat the last one
                const int yr = gr.yrow_of[(size_t)d * ng + gi];
                const long long e = dly(d, gi * G) - h.sigma[dle];
                add_use(u.blk, yr, e);
                add_use(u.quad[dl / DQ], yr, e);
            }
            for (int q = 0; q < 4; ++q) {
                u.cols[q] = u.chunks[q] = 0;
                for (const Use &x : u.quad[q]) {
                    const int c8 = (int)ceil_to(16 + (x.emax - x.emin), 8);      // the consumers load 16 columns
                    u.cols[q] += c8;
                    u.chunks[q] += (c8 + 15) / 16;                                // staged 16 columns at a time (+ one 8)
                }
                if (u.cols[q] > kTmCols || u.chunks[q] > kTmCQMax) return false;
            }
            if (u.blk.size() > 32) return false;
            for (const Use &x : u.blk) need_max = std::max(need_max, x.emax - floor_to(x.emin, al) + span);
        }
    const int pitch = (int)ceil_to(need_max, al) + 16;       // + 16: the stagers read whole 8-column chunks of 16 + S columns
    // greedy packing of consecutive groups into slabs
    struct Slab { int g0, g1; };
    std::vector<std::vector<Slab>> slabs(nblk);
    int cs_max = 0, nslab_max = 0;
    long long ngroups_total = 0, nslabs_total = 0;
    double cols_total = 0;
    for (int blk = 0; blk < nblk; ++blk) {
        int g0 = 0;
        while (g0 < ng) {
            int rows = 0, cols[4] = {0, 0, 0, 0}, nrq[4] = {0, 0, 0, 0}, g1 = g0;
            while (g1 < ng && g1 - g0 < kTmQMax) {
                const GroupUse &u = gu[blk][g1];
                bool fits = rows + (int)u.blk.size() <= 32;
                for (int q = 0; q < 4; ++q) fits = fits && cols[q] + u.cols[q] <= kTmCols && nrq[q] + u.chunks[q] <= kTmCQMax;
                if (!fits) break;
                rows += (int)u.blk.size();
                for (int q = 0; q < 4; ++q) { cols[q] += u.cols[q]; nrq[q] += u.chunks[q]; cols_total += u.cols[q]; }
                ++g1;
            }
            if (g1 == g0) return false;
            cs_max = std::max(cs_max, rows);
            slabs[blk].push_back({g0, g1});
            g0 = g1;
        }
        nslab_max = std::max(nslab_max, (int)slabs[blk].size());
        ngroups_total += ng;
        nslabs_total += (long long)slabs[blk].size();
    }
    const int CS = cs_max;
    const size_t stage = (((size_t)CS * pitch * 4 + (size_t)tabw * 4) + 127) & ~(size_t)127;
    const size_t fixed = (size_t)2 * 16 * kTmEnt * 4 + 320;                  // entry copies, barriers, TMEM base slot
    const int stages = (int)std::min<size_t>(8, (kSmemBudget - fixed - 64) / stage);
    if (stages < 2) return false;
    h.rowdesc.assign((size_t)nblk * nslab_max * CS, make_int4(-1, 0, 0, 0));
    h.tab.assign((size_t)nblk * nslab_max * tabw, 0u);
    h.nslab.resize(nblk);
    for (int blk = 0; blk < nblk; ++blk) {
        h.nslab[blk] = (int32_t)slabs[blk].size();
        for (size_t s = 0; s < slabs[blk].size(); ++s) {
            int4 *rd = &h.rowdesc[((size_t)blk * nslab_max + s) * CS];
            uint32_t *tab = &h.tab[((size_t)blk * nslab_max + s) * tabw];
            int r = 0, nrq[4] = {0, 0, 0, 0}, tcol[4] = {0, 0, 0, 0};
            tab[4] = (uint32_t)(slabs[blk][s].g1 - slabs[blk][s].g0);
            for (int gi = slabs[blk][s].g0; gi < slabs[blk][s].g1; ++gi) {
                const GroupUse &u = gu[blk][gi];
                const int qi = gi - slabs[blk][s].g0;
                for (size_t k = 0; k < u.blk.size(); ++k) {
                    const long long rs = floor_to(u.blk[k].emin, al);
                    rd[r + k] = make_int4(u.blk[k].yrow, (int)rs, (int)ceil_to(u.blk[k].emax - rs + span, al), 0);
                }
                for (int q = 0; q < 4; ++q) {
                    std::vector<int> col_of(u.quad[q].size());
                    for (size_t k = 0; k < u.quad[q].size(); ++k) {
                        const Use &x = u.quad[q][k];
                        size_t kb = 0;
                        while (u.blk[kb].yrow != x.yrow) ++kb;
                        const long long rs = floor_to(u.blk[kb].emin, al);
                        int n8 = (int)ceil_to(16 + (x.emax - x.emin), 8) / 8;
                        col_of[k] = tcol[q];
                        uint32_t soff = (uint32_t)((long long)(r + kb) * pitch + (x.emin - rs));
                        while (n8 > 0) {                                          // chunks of 16 columns, then one of 8
                            const int c = n8 >= 2 ? 2 : 1;
                            const int slot = nrq[q]++;
                            tab[8 + (q * kTmCQMax + slot) * 2] = soff;
                            tab[8 + (q * kTmCQMax + slot) * 2 + 1] = (uint32_t)tcol[q] | ((uint32_t)(c - 1) << 16);
                            soff += 8 * c;
                            tcol[q] += 8 * c;
                            n8 -= c;
                        }
                    }
                    for (int dq = 0; dq < DQ; ++dq) {
                        const int dl = q * DQ + dq;
                        const int d = std::min(blk * DB + dl, p->ndms - 1), dle = d - blk * DB;
                        const int yr = gr.yrow_of[(size_t)d * ng + gi];
                        size_t k = 0;
                        while (u.quad[q][k].yrow != yr) ++k;
                        const long long e = dly(d, gi * G) - h.sigma[dle];
                        tab[8 + 4 * kTmCQMax * 2 + (size_t)dl * kTmQMax + qi] = (uint32_t)(col_of[k] + (e - u.quad[q][k].emin));
                    }
                }
                r += (int)u.blk.size();
            }
            for (int q = 0; q < 4; ++q) tab[q] = (uint32_t)nrq[q];
        }
    }
    tt.D = D; tt.P = P; tt.DB = DB; tt.span = span; tt.CS = CS; tt.pitch = pitch; tt.stages = stages;
    tt.nslab_max = nslab_max; tt.nblk = nblk; tt.tabw = tabw;
    tt.sigma_max = *std::max_element(h.sigma.begin(), h.sigma.end());
    tt.smem_bytes = (size_t)stages * stage + fixed;
    tt.groups_per_slab = (double)ngroups_total / (double)nslabs_total;
    tt.cols_per_group = cols_total / (4.0 * (double)ngroups_total);
    return true;
}

static void free_tmem_tables(TmemTables *tt)
{
    cudaFree(tt->d_rowdesc); cudaFree(tt->d_tab); cudaFree(tt->d_nslab); cudaFree(tt->d_sigma);
    *tt = TmemTables();
}

static void free_rows_tables(RowsTables *rt)
{
    cudaFree(rt->d_rowdesc); cudaFree(rt->d_ent); cudaFree(rt->d_sigma); cudaFree(rt->d_group_row0); cudaFree(rt->d_ydelta);
    *rt = RowsTables();
}

// Modelled cost of a group size in units of one shared-memory operand word per output sample: nchans/G words in the
// main kernel, plus the y rows, each written to and read back from HBM.  Measured on B200 (cfg 3 and cfg 5, G = 4..8): a
// row and sample costs about 7 word-times at the HBM copy rate; 11 also covers the slabs getting shorter (more rows per
// group) as G grows, and reproduces the measured optimum (G = 5 at 1024 channels x 640 DMs, 6-7 at 4096 x 2048).
// The packed 16-bit kernel (uint8 / 4-bit input) is bound by issue slots rather than by operand words and gains less
// from wider groups: measured optimum G = 4 on cfg 4 (9.75 ms; G = 5: 10.8, G = 6: 12.3), hence the larger weight.
static double group_cost(const mdsm_plan *p, const GroupRows &gr, bool packed16)
{
    return (double)p->ndms * gr.ngroups + (packed16 ? 16.0 : 11.0) * gr.nyrows;
}

// Dynamic shared memory of the pre-pass (group_presum_*): G rows of chunk + dmax samples in the input's element type, then
// the group's pattern table.  kind 0: 32-bit samples (MDSM_F32, MDSM_U16), 1: uint8, 2: 4-bit.  delta_off = where the
// pattern table starts.  Used at plan time (a group size that does not fit is skipped) and at launch time.
constexpr size_t kPreSmemLimit = 200 * 1024;
static size_t presum_smem_bytes(int kind, int G, int dmax, int maxpat, size_t *delta_off)
{
    const int chunk = kind == 0 ? kPreChunkF32 : kPreChunkU8;
    const size_t rows = kind == 0 ? (size_t)G * (chunk + dmax) * 4
                                  : (kind == 1 ? (size_t)G * (chunk + ((dmax + 3) & ~3) + 4) : (size_t)G * ((((chunk + dmax) / 2 + 3) & ~3) + 8));
    const size_t off = (rows + 15) & ~(size_t)15;
    if (delta_off) *delta_off = off;
    return off + (size_t)maxpat * kGMax * sizeof(int16_t);
}

static int build_dtype(mdsm_plan *p, int kind /* 0: 32-bit rows, 1: uint8 -> 16-bit rows, 2: 4-bit -> 16-bit rows */, const std::vector<GroupRows> &cands)
{
    const bool f32 = kind == 0;
    RowsTables &rt = kind == 0 ? p->rows_f32 : (kind == 1 ? p->rows_u8 : p->rows_u4);
    free_rows_tables(&rt);
    if (f32) free_tmem_tables(&p->tmem_f32);
    const RowsGeom geom = f32 ? kGeomRowsF32 : kGeomRowsU16;
    // candidates in the order of their modelled cost; the first whose tables fit the kernel's limits is taken
    std::vector<const GroupRows *> order;
    for (const GroupRows &gr : cands) order.push_back(&gr);
    std::sort(order.begin(), order.end(), [&](const GroupRows *x, const GroupRows *y) { return group_cost(p, *x, !f32) < group_cost(p, *y, !f32); });
    for (const GroupRows *gr : order) {
        RowsHost h;
        if (!build_rows_tables(p, f32, kind == 2 ? kPartChansU4 : kPartChansU8, *gr, geom, rt, h)) continue;
        // the pre-pass of this group size must fit its shared memory too, or every mdsm_dedisperse would fail at launch
        // although kernel_info says "rows": try the next candidate (a smaller G has a smaller delay range per group)
        if (presum_smem_bytes(kind, rt.G, rt.dmax, rt.maxpat, nullptr) > kPreSmemLimit) { rt = RowsTables(); continue; }
        if (!upload((int4 **)&rt.d_rowdesc, h.rowdesc) || !upload(&rt.d_ent, h.ent) || !upload(&rt.d_sigma, h.sigma) ||
            !upload(&rt.d_group_row0, gr->group_row0) || !upload(&rt.d_ydelta, gr->ydelta)) {
            mdsm_set_error("dedispersion table upload failed: %s", cudaGetErrorString(cudaGetLastError()));
            free_rows_tables(&rt);
            return MDSM_ECUDA;
        }
        rt.ok = true;
        if (f32) {
            // the TMEM variant of the main kernel shares the pre-pass, the scratch layout and the group size
            free_tmem_tables(&p->tmem_f32);
            TmemHost th;
            TmemTables &tt = p->tmem_f32;
            if (build_tmem_tables(p, *gr, tt, th)) {
                if (!upload((int4 **)&tt.d_rowdesc, th.rowdesc) || !upload(&tt.d_tab, th.tab) || !upload(&tt.d_nslab, th.nslab) ||
                    !upload(&tt.d_sigma, th.sigma)) {
                    mdsm_set_error("dedispersion table upload failed: %s", cudaGetErrorString(cudaGetLastError()));
                    free_tmem_tables(&tt);
                    return MDSM_ECUDA;
                }
                tt.ok = true;
            }
        }
        return MDSM_OK;
    }
    return MDSM_OK;                                                    // no table: the direct kernel runs
}

template <int G> static cudaError_t launch_presum(int dtype, const PreArgs &a, dim3 grid, size_t smem, cudaStream_t st)
{
    cudaError_t e = cudaSuccess;
    // only very wide groups need more than the default dynamic shared memory; set per launch (per-device state)
    if (dtype == MDSM_F32) {
        if (smem > 48 * 1024) e = cudaFuncSetAttribute(group_presum_w32_kernel<G, float, float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) group_presum_w32_kernel<G, float, float><<<grid, kPreThreads, smem, st>>>(a);
    } else if (dtype == MDSM_U16) {
        if (smem > 48 * 1024) e = cudaFuncSetAttribute(group_presum_w32_kernel<G, uint16_t, uint32_t>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) group_presum_w32_kernel<G, uint16_t, uint32_t><<<grid, kPreThreads, smem, st>>>(a);
    } else if (dtype == MDSM_U8) {
        if (smem > 48 * 1024) e = cudaFuncSetAttribute(group_presum_u8_kernel<G>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) group_presum_u8_kernel<G><<<grid, kPreThreads, smem, st>>>(a);
    } else {
        if (smem > 48 * 1024) e = cudaFuncSetAttribute(group_presum_u4_kernel<G>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) group_presum_u4_kernel<G><<<grid, kPreThreads, smem, st>>>(a);
    }
    return e;
}

template <typename Tr> static int launch_rows(const RowsArgs &a, size_t smem, int grid, cudaStream_t st)
{
    auto kern = dedisperse_rows_kernel<Tr>;
    // per launch: the attribute belongs to the current device's copy of the kernel, and the call costs microseconds
    MDSM_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    kern<<<grid, (Tr::NW + 1) * 32, smem, st>>>(a);
    MDSM_CUDA_TRY(cudaGetLastError());
    return MDSM_OK;
}

}  // namespace

int mdsm_rows_build_tables(mdsm_plan *p)
{
    std::vector<GroupRows> cands;
    for (int G = 1; G <= kGMax; ++G) {
        if (p->group_size > 0 && G != p->group_size) continue;
        GroupRows gr;
        if (enumerate_group_rows(p, G, gr)) cands.push_back(std::move(gr));
    }
    int rc = build_dtype(p, 0, cands);
    if (rc == MDSM_OK) rc = build_dtype(p, 1, cands);
    if (rc == MDSM_OK) rc = build_dtype(p, 2, cands);
    return rc;
}

void mdsm_rows_free_tables(mdsm_plan *p)
{
    free_tmem_tables(&p->tmem_f32);
    free_rows_tables(&p->rows_f32);
    free_rows_tables(&p->rows_u8);
    free_rows_tables(&p->rows_u4);
}

size_t mdsm_rows_scratch_bytes_per_beam(const mdsm_plan *p, int dtype)
{
    const RowsTables &rt = mdsm_rows_of(p, dtype);
    return rt.ok ? (size_t)rt.nyrows * (size_t)rt.ystride * ((dtype == MDSM_F32 || dtype == MDSM_U16) ? 4 : 2) : 0;
}

int mdsm_launch_dedisperse_rows(mdsm_plan *p, const void *d_in, int dtype, int beam0, int nb, void *d_out, cudaStream_t st)
{
    const bool f32 = dtype == MDSM_F32, w32 = dtype == MDSM_F32 || dtype == MDSM_U16;
    const RowsTables &rt = mdsm_rows_of(p, dtype);
    void *scratch = p->d_scratch[dtype];
    const int nslots = p->scratch_slots[dtype];
    MDSM_REQUIRE(rt.ok && scratch && nslots >= 1, "dedispersion scratch not reserved (call mdsm_plan_reserve)");
    const int ntile_t = (int)((p->nsamps_out + rt.sigma_max + rt.stride - 1) / rt.stride);
    const int chunk = w32 ? kPreChunkF32 : kPreChunkU8;
    size_t delta_off = 0;
    const size_t pre_smem_all = presum_smem_bytes(w32 ? 0 : (dtype == MDSM_U8 ? 1 : 2), rt.G, rt.dmax, rt.maxpat, &delta_off);
    MDSM_REQUIRE(pre_smem_all <= kPreSmemLimit, "pre-pass: group delay range or pattern count too large");   // plan time excludes it
    // beams go through the scratch `nslots` at a time (slot = beam % nslots), in stream order
    for (int bs = beam0; bs < beam0 + nb; bs += nslots) {
        const int n = std::min(nslots, beam0 + nb - bs);
        PreArgs pa;
        pa.in = d_in; pa.y = scratch; pa.group_row0 = rt.d_group_row0; pa.ydelta = rt.d_ydelta;
        pa.beam0 = bs; pa.nslots = nslots; pa.nchans = p->nchans; pa.G = rt.G; pa.nyrows = rt.nyrows; pa.dmax = rt.dmax;
        pa.nsamps = p->nsamps; pa.ystride = rt.ystride; pa.delta_off = (int)delta_off;
        dim3 grid((unsigned)((rt.ystride + chunk - 1) / chunk), rt.ngroups, n);
        MDSM_REQUIRE(rt.ngroups <= 65535 && n <= 65535, "pre-pass: grid too large");
        cudaError_t pe;
        switch (rt.G) {
            case 1: pe = launch_presum<1>(dtype, pa, grid, pre_smem_all, st); break;
            case 2: pe = launch_presum<2>(dtype, pa, grid, pre_smem_all, st); break;
            case 3: pe = launch_presum<3>(dtype, pa, grid, pre_smem_all, st); break;
            case 4: pe = launch_presum<4>(dtype, pa, grid, pre_smem_all, st); break;
            case 5: pe = launch_presum<5>(dtype, pa, grid, pre_smem_all, st); break;
            case 6: pe = launch_presum<6>(dtype, pa, grid, pre_smem_all, st); break;
            case 7: pe = launch_presum<7>(dtype, pa, grid, pre_smem_all, st); break;
            default: pe = launch_presum<8>(dtype, pa, grid, pre_smem_all, st); break;
        }
        MDSM_CUDA_TRY(pe);
        MDSM_CUDA_TRY(cudaGetLastError());
        p->launches += 1;

        int rc;
        const TmemTables &tt = p->tmem_f32;
        if (f32 && tt.ok && p->dedisp_kernel == 3) {          // experimental variant: only on request
            TmemArgs a;
            a.y = (const float *)scratch; a.out = (float *)d_out;
            a.rowdesc = (const int4 *)tt.d_rowdesc; a.tab = tt.d_tab; a.nslab = tt.d_nslab; a.sigma = tt.d_sigma;
            a.beam0 = bs; a.nslots = nslots; a.nyrows = rt.nyrows; a.ndms = p->ndms;
            a.nblk = tt.nblk; a.ntile_t = (int)((p->nsamps_out + tt.sigma_max + tt.span - 1) / tt.span);
            a.nslab_max = tt.nslab_max; a.CS = tt.CS; a.pitch = tt.pitch; a.stages = tt.stages; a.tabw = tt.tabw; a.span = tt.span;
            a.ntiles = (long long)tt.nblk * a.ntile_t * n;
            a.nsamps = p->nsamps; a.nsamps_out = p->nsamps_out; a.ystride = rt.ystride;
            auto kern = dedisperse_tmem_kernel<kGeomTmem.D, kGeomTmem.P>;
            MDSM_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tt.smem_bytes));
            kern<<<(int)std::min<long long>(a.ntiles, p->sm_count), kTmWarps * 32, tt.smem_bytes, st>>>(a);
            MDSM_CUDA_TRY(cudaGetLastError());
            rc = MDSM_OK;
        } else {
        RowsArgs a;
        a.y = scratch; a.out = d_out;
        a.rowdesc = (const int4 *)rt.d_rowdesc; a.ent = rt.d_ent; a.sigma = rt.d_sigma;
        a.beam0 = bs; a.nslots = nslots; a.nyrows = rt.nyrows; a.ndms = p->ndms;
        a.nblk = rt.nblk; a.ntile_t = ntile_t; a.nslab = rt.nslab; a.Q = rt.Q; a.ngroups = rt.ngroups; a.CS = rt.CS;
        a.pitch = rt.pitch; a.stages = rt.stages; a.slabs_per_part = rt.slabs_per_part; a.stride = rt.stride;
        a.ntiles = (long long)rt.nblk * ntile_t * n;
        a.nsamps = p->nsamps; a.nsamps_out = p->nsamps_out; a.ystride = rt.ystride;
        const int grid_main = (int)std::min<long long>(a.ntiles, p->sm_count);
        if (f32) rc = launch_rows<RowsTraits<kGeomRowsF32.D, kGeomRowsF32.T, kGeomRowsF32.NW, true>>(a, rt.smem_bytes, grid_main, st);
        else if (w32) rc = launch_rows<RowsTraits<kGeomRowsF32.D, kGeomRowsF32.T, kGeomRowsF32.NW, true, true>>(a, rt.smem_bytes, grid_main, st);
        else rc = launch_rows<RowsTraits<kGeomRowsU16.D, kGeomRowsU16.T, kGeomRowsU16.NW, false>>(a, rt.smem_bytes, grid_main, st);
        }
        if (rc != MDSM_OK) return rc;
        p->launches += 1;
    }
    return MDSM_OK;
}
