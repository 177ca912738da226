// Tiled brute-force dedispersion for sm_100a (BASELINE.json north_star item 2).
//
//   out[b][d][t] = sum_c in[b][c][t + delay(d,c)]
//
// Work decomposition:
//   tile  = one beam x one block of DB = NW*D consecutive DM trials x one time tile of 32*T samples.
//   CTA   = persistent: one per SM, walks tiles (DM block fastest, so that the CTAs running together
//           read the same input rows out of L2) and, inside a tile, the channel PARTS (u8 only: <= 256
//           channels, the most a 16-bit lane can hold) and the channel SLABS of a part.
//   warp  = D consecutive DM trials of the block, all 32*T samples of the tile.
//   thread= D x T accumulators in registers: T CONSECUTIVE samples (lane*T ...) of each of its D DMs.
// Per channel a thread loads ONE register window of T + (spread of its D delays) consecutive samples
// from shared memory with conflict-free 128-bit loads and adds it, at D different register offsets, into
// its D accumulator rows -- every shared-memory word feeds ~3 adds, which is what lifts the kernel off the
// 32 words/clk/SM shared-memory ceiling (25 % of the add peak).  The offsets are warp-uniform; they select
// straight-line add blocks, chained through short trees of direct conditional branches (chain_gen.h, gen_chain.py).
//   fp32: accumulators and window are packed f32x2 register pairs (FADD2 for even offsets).
//   u8  : the input is widened once to u16 (plan scratch); accumulators are packed u16x2 lanes (one add =
//         two samples), flushed into the uint32 output after every part (part 0 stores, later parts
//         read-modify-write their own elements, which are still in L2).  Every DM keeps an even-phase and an
//         odd-phase accumulator row, so that odd register offsets need no shifted copy of the window.
// The time axis is SHEARED: DM d of a block owns outputs [tile_t0 - sigma_d, tile_t0 - sigma_d + 32T)
// with sigma_d ~ half the band-edge delay slope, which halves the spread of the D windows (and of the
// staged rows) compared with an unsheared tile.
// Staging: a producer warp streams channel slabs (CS rows of `row_elems` samples, each starting at its own
// 16-byte-aligned delay-dependent offset) into a ring of shared-memory stages with 1-D TMA bulk copies
// (cp.async.bulk ... mbarrier::complete_tx), full/empty mbarriers per stage; it runs ahead across tile
// boundaries, so a CTA never drains its pipeline between tiles.
#include <algorithm>
#include <cmath>
#include <vector>

#include "chain_gen.h"
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
// producer-side wait: the producer runs several stages ahead, so it sleeps between polls instead of
// spinning (a spinning producer warp took 12 % of the SM's issue slots in the r1b profile)
__device__ __forceinline__ void mbar_wait_sleep(uint64_t *bar, uint32_t parity)
{
    while (!mbar_try_wait(bar, parity)) __nanosleep(2000);
}
__device__ __forceinline__ void bulk_g2s(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// Writes v[0..T) to orow[ts .. ts+T), clipped to [0, n); ACCUM adds to what is there (the elements are
// this thread's own: no other thread of the launch touches them).  Rows are 16-byte aligned; ts is not (the
// shear is a whole number of samples), so the head up to the next multiple of 4 goes out as scalars and the
// rest as 128-bit accesses.  The head length is warp-uniform: one switch, static register indexing.
template <int T, int H, bool ACCUM, typename V>
__device__ __forceinline__ void store_row_h(V *orow, long long ts, long long n, const V (&v)[T])
{
#pragma unroll
    for (int i = 0; i < H; ++i)
        if (ts + i >= 0 && ts + i < n) orow[ts + i] = ACCUM ? (V)(orow[ts + i] + v[i]) : v[i];
#pragma unroll
    for (int i = H; i + 3 < T; i += 4) {
        const long long t = ts + i;
        if (t >= 0 && t + 3 < n) {
            uint4 q;
            q.x = reinterpret_cast<const uint32_t &>(v[i]); q.y = reinterpret_cast<const uint32_t &>(v[i + 1]);
            q.z = reinterpret_cast<const uint32_t &>(v[i + 2]); q.w = reinterpret_cast<const uint32_t &>(v[i + 3]);
            if (ACCUM) {                                   // integer path only (uint32 adds)
                const uint4 o = *reinterpret_cast<const uint4 *>(orow + t);
                q.x += o.x; q.y += o.y; q.z += o.z; q.w += o.w;
            }
            *reinterpret_cast<uint4 *>(orow + t) = q;
        } else {
#pragma unroll
            for (int k = 0; k < 4; ++k)
                if (t + k >= 0 && t + k < n) orow[t + k] = ACCUM ? (V)(orow[t + k] + v[i + k]) : v[i + k];
        }
    }
#pragma unroll
    for (int i = H + (T - H) / 4 * 4; i < T; ++i)
        if (ts + i >= 0 && ts + i < n) orow[ts + i] = ACCUM ? (V)(orow[ts + i] + v[i]) : v[i];
}
template <int T, bool ACCUM, typename V>
__device__ __forceinline__ void store_row(V *orow, long long ts, long long n, const V (&v)[T])
{
    static_assert(sizeof(V) == 4, "32-bit outputs");
    switch ((int)((4 - (ts & 3)) & 3)) {
        case 0: store_row_h<T, 0, ACCUM>(orow, ts, n, v); break;
        case 1: store_row_h<T, 1, ACCUM>(orow, ts, n, v); break;
        case 2: store_row_h<T, 2, ACCUM>(orow, ts, n, v); break;
        default: store_row_h<T, 3, ACCUM>(orow, ts, n, v); break;
    }
}

// tile index -> (DM block, time tile, beam); DM block fastest
struct TileWalk {
    int nblk, ntile_t;
    long long ntiles;
    __device__ __forceinline__ void decode(long long tile, int &blk, int &tt, int &bb) const
    {
        blk = (int)(tile % nblk);
        const long long rest = tile / nblk;
        tt = (int)(rest % ntile_t);
        bb = (int)(rest / ntile_t);
    }
};

struct TiledArgs {
    const void *in;
    void *out;
    const int32_t *row_start;             // [nblk][nslab*CS]  first staged sample of the row, relative to tile_t0
    const unsigned long long *warp_tab;   // [nblk][nslab][NW][CS] window entries (format: gen_chain.py)
    const int32_t *sigma;                 // [DB] output time shear per DM of a block
    const int32_t *src_row;               // pair mode: [nblk][nslab*CS] source row of staged row r (-1: none); else nullptr
    const int32_t *nslab_blk;             // pair mode: [nblk] slabs of the block; else nullptr
    int nrows_src;                        // rows per beam of the staged source (nchans, or the pre-summed copy's row count)
    int nparts;                           // pair mode: parts per tile (slabs per part = the block's slabs / nparts); else 0
    int beam0, nchans, nslab, slabs_per_part, ndms;
    long long nsamps, nsamps_out;
    int row_elems, stages;
    TileWalk walk;
};

template <int D_, int T_, int NW_, int CS_, int NOFF_> struct TraitsF32 {
    static constexpr int D = D_, T = T_, NW = NW_, CS = CS_, AW = T_ / 2;
    static constexpr bool kF32 = true, kTwoPhase = false, kPairs = false;
    static constexpr int PW = NW_ % 4 == 0 ? 4 : 1;     // producer warpgroup (register reallocation) or one producer warp
    using In = float; using Out = float; using Acc = unsigned long long;
    using Slab = SlabF32<D_, T_, NOFF_>;
    static_assert(T_ % 4 == 0 && (T_ / 4) % 2 == 1, "T/4 must be odd (bank-conflict-free 128-bit window loads)");
};
// pair pre-sum mode: same data types as TraitsF32, loop with skip bits and per-slot dispatchers (gen_chain.py: gen_f32p)
template <int D_, int T_, int NW_, int CS_, int NOFF_> struct TraitsF32P : TraitsF32<D_, T_, NW_, CS_, NOFF_> {
    static constexpr bool kPairs = true;
    using Slab = SlabF32P<D_, T_, NOFF_>;
};
template <int D_, int T_, int NW_, int CS_, int NOFF_> struct TraitsU16 {
    static constexpr int D = D_, T = T_, NW = NW_, CS = CS_, AW = T_ / 2;
    static constexpr bool kF32 = false, kTwoPhase = false, kPairs = false;
    static constexpr int PW = 1;
    using In = uint16_t; using Out = uint32_t; using Acc = unsigned;
    using Slab = SlabU16<D_, T_, NOFF_>;
    static_assert(T_ % 8 == 0 && (T_ / 8) % 2 == 1, "T/8 must be odd (bank-conflict-free 128-bit window loads)");
};

// two-phase integer variant: per DM an even-phase row E (T/2 registers) and an odd-phase row O (T/2 + 1 registers,
// outputs shifted by one sample), no shifted window copy (gen_chain.py: gen_u16p)
template <int D_, int T_, int NW_, int CS_, int NOFF_> struct TraitsU16P {
    static constexpr int D = D_, T = T_, NW = NW_, CS = CS_, AW = T_ + 1;
    static constexpr bool kF32 = false, kTwoPhase = true, kPairs = false;
    static constexpr int PW = 1;
    using In = uint16_t; using Out = uint32_t; using Acc = unsigned;
    using Slab = SlabU16P<D_, T_, NOFF_>;
    static_assert(T_ % 8 == 0 && (T_ / 8) % 2 == 1, "T/8 must be odd (bank-conflict-free 128-bit window loads)");
};

// integer pair pre-sum mode: TraitsU16P's data layout, loop with skip bits (gen_chain.py: gen_u16pp)
template <int D_, int T_, int NW_, int CS_, int NOFF_> struct TraitsU16PP : TraitsU16P<D_, T_, NW_, CS_, NOFF_> {
    static constexpr bool kPairs = true;
    using Slab = SlabU16PP<D_, T_, NOFF_>;
};

// ------------------------------------------------------------------ the kernel
template <typename Tr>
__global__ void __launch_bounds__((Tr::NW + Tr::PW) * 32, 1) dedisperse_tiled_kernel(const TiledArgs a)
{
    using In = typename Tr::In;
    using Out = typename Tr::Out;
    using Acc = typename Tr::Acc;
    constexpr int D = Tr::D, T = Tr::T, NW = Tr::NW, CS = Tr::CS, AW = Tr::AW, DB = D * NW;
    static_assert(CS <= 31, "producer lanes 0..CS-1 copy rows, lane CS the table slice");
    extern __shared__ __align__(128) unsigned char smem[];
    const int stages = a.stages;
    const uint32_t stage_bytes = (uint32_t)CS * a.row_elems * sizeof(In);
    unsigned long long *tabs = reinterpret_cast<unsigned long long *>(smem + (size_t)stages * stage_bytes);
    uint64_t *full = reinterpret_cast<uint64_t *>(tabs + (size_t)stages * NW * CS);
    uint64_t *empty = full + stages;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    // Rows that stick out of [0, nsamps) are only partly written by the bulk copies.  What they leave behind
    // feeds outputs outside [0, nsamps_out) only, but a stale 16-bit lane must never carry into its valid
    // neighbour: with the stages zeroed once, every staged value is zero or a real sample.
    for (uint32_t i = threadIdx.x; i < stages * stage_bytes / 16; i += blockDim.x) reinterpret_cast<uint4 *>(smem)[i] = make_uint4(0, 0, 0, 0);
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    if (threadIdx.x == 0) {
        for (int s = 0; s < stages; ++s) {
            mbar_init(&full[s], CS + 1);
            mbar_init(&empty[s], NW);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const int ncp = a.nslab * CS;
    if (warp >= NW) {
        // NW % 4 == 0: the producer owns a whole warpgroup and hands its registers to the consumers
        if constexpr (Tr::PW == 4) asm volatile("setmaxnreg.dec.sync.aligned.u32 24;");
        if (warp > NW) return;
        // ===== producer: lane r < CS copies row r of every slab, lane CS the slab's slice of the warp table =====
        if (lane > CS) return;
        int st = 0;
        uint32_t ph = 1;             // parity of the empty-barrier phase to wait for (first lap: no wait)
        bool first_lap = true;
        for (long long tile = blockIdx.x; tile < a.walk.ntiles; tile += gridDim.x) {
            int blk, tt, bb;
            a.walk.decode(tile, blk, tt, bb);
            const long long tile_t0 = (long long)tt * (32 * T);
            const In *beam_in = reinterpret_cast<const In *>(a.in) + (size_t)(a.beam0 + bb) * a.nrows_src * (size_t)a.nsamps;
            const int32_t *rs = a.row_start + (size_t)blk * ncp;
            const int32_t *sr = Tr::kPairs ? a.src_row + (size_t)blk * ncp : nullptr;
            const unsigned long long *wt = a.warp_tab + (size_t)blk * a.nslab * NW * CS;
            const int nslab_b = Tr::kPairs ? a.nslab_blk[blk] : a.nslab;
            for (int slab = 0; slab < nslab_b; ++slab) {
                if (!first_lap) mbar_wait_sleep(&empty[st], ph);
                if (lane < CS) {
                    const int r = slab * CS + lane;
                    const int c = Tr::kPairs ? sr[r] : (r < a.nchans ? r : -1);      // source row of staged row r
                    uint32_t bytes = 0;
                    long long lo = 0, g0 = 0;
                    if (c >= 0) {
                        g0 = tile_t0 + rs[r];
                        lo = g0 < 0 ? 0 : g0;
                        long long hi = g0 + a.row_elems;
                        if (hi > a.nsamps) hi = a.nsamps;
                        if (hi > lo) bytes = (uint32_t)((hi - lo) * sizeof(In));
                    }
                    mbar_arrive_expect_tx(&full[st], bytes);
                    if (bytes)
                        bulk_g2s(smem + (size_t)st * stage_bytes + ((size_t)lane * a.row_elems + (lo - g0)) * sizeof(In),
                                 beam_in + (size_t)c * a.nsamps + lo, bytes, &full[st]);
                } else {
                    const uint32_t bytes = NW * CS * sizeof(unsigned long long);
                    mbar_arrive_expect_tx(&full[st], bytes);
                    bulk_g2s(tabs + (size_t)st * NW * CS, wt + (size_t)slab * NW * CS, bytes, &full[st]);
                }
                if (++st == stages) { st = 0; ph ^= 1; first_lap = false; }
            }
        }
        return;
    }

    // ===== consumer warps =====
    if constexpr (Tr::PW == 4) asm volatile("setmaxnreg.inc.sync.aligned.u32 160;");
    Acc acc[D][AW];
    const uint32_t lane_base = smem_u32(smem) + lane * (T * (uint32_t)sizeof(In));
    const uint32_t tab_base = smem_u32(tabs) + warp * (CS * 8);
    int st = 0;
    uint32_t ph = 0;
    for (long long tile = blockIdx.x; tile < a.walk.ntiles; tile += gridDim.x) {
        int blk, tt, bb;
        a.walk.decode(tile, blk, tt, bb);
        const long long tile_t0 = (long long)tt * (32 * T);
        const int b = a.beam0 + bb;
#pragma unroll 1
        const int nslab_b = Tr::kPairs ? a.nslab_blk[blk] : a.nslab;
        const int spp = !Tr::kPairs ? a.slabs_per_part : (Tr::kF32 ? nslab_b : nslab_b / a.nparts);   // fp32 tiles have one part
#pragma unroll 1
        for (int s0 = 0; s0 < nslab_b; s0 += spp) {
#pragma unroll
            for (int j = 0; j < D; ++j)
#pragma unroll
                for (int i = 0; i < AW; ++i) acc[j][i] = 0;      // (+0.f, +0.f) / (0, 0)
            const int s1 = min(nslab_b, s0 + spp);
#pragma unroll 1
            for (int slab = s0; slab < s1; ++slab) {
                mbar_wait(&full[st], ph);
                Tr::Slab::run(acc, lane_base + st * stage_bytes, tab_base + st * (NW * CS * 8));
                __syncwarp();
                if (lane == 0) mbar_arrive(&empty[st]);
                if (++st == stages) { st = 0; ph ^= 1; }
            }
            // ----- epilogue of the part: each thread owns T consecutive outputs of each of its D DMs -----
#pragma unroll
            for (int j = 0; j < D; ++j) {
                const int dl = warp * D + j;
                const int d = blk * DB + dl;
                if (d >= a.ndms) continue;
                Out v[T];
#pragma unroll
                for (int i = 0; i < T / 2; ++i) {
                    if constexpr (Tr::kTwoPhase) {
                        v[2 * i] = (acc[j][i] & 0xffffu) + (acc[j][T / 2 + i] >> 16);
                        v[2 * i + 1] = (acc[j][i] >> 16) + (acc[j][T / 2 + i + 1] & 0xffffu);
                    } else if constexpr (Tr::kF32) {
                        v[2 * i] = __uint_as_float((unsigned)acc[j][i]);
                        v[2 * i + 1] = __uint_as_float((unsigned)(acc[j][i] >> 32));
                    } else {
                        v[2 * i] = acc[j][i] & 0xffffu;
                        v[2 * i + 1] = acc[j][i] >> 16;
                    }
                }
                const long long ts = tile_t0 - a.sigma[dl] + (long long)lane * T;
                Out *orow = reinterpret_cast<Out *>(a.out) + ((size_t)b * a.ndms + d) * (size_t)a.nsamps;
                if (Tr::kF32 || s0 == 0) store_row<T, false>(orow, ts, a.nsamps_out, v);
                else store_row<T, true>(orow, ts, a.nsamps_out, v);
            }
        }
    }
}

// widens the uint8 filterbank to uint16 (the staged element type of the integer kernels), 8 samples per thread and
// step (nsamps % 8 == 0 is a condition of the tiled integer path, so every beam is a whole number of such groups)
__global__ void __launch_bounds__(256) widen_u8_kernel(const uint2 *__restrict__ in, uint4 *__restrict__ out, size_t n8)
{
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n8; i += (size_t)gridDim.x * blockDim.x) {
        const uint2 v = in[i];
        uint4 a;
        a.x = __byte_perm(v.x, 0, 0x4140); a.y = __byte_perm(v.x, 0, 0x4342);
        a.z = __byte_perm(v.y, 0, 0x4140); a.w = __byte_perm(v.y, 0, 0x4342);
        out[i] = a;
    }
}

// Pair pre-sum (fp32): y[row][t] = x[c][t] + x[c+1][t + delta], row = (channel pair (c, c+1), delay difference delta).
// delay(d, c+1) - delay(d, c) takes few values over the DM grid, so out[d][t] = sum over pairs of
// y[(pair, delta(d, pair))][t + delay(d, c)]: the same terms, added two at a time.  One CTA column per pair writes all
// the rows of that pair (consecutive in y), so x is read once.
__global__ void __launch_bounds__(256) pair_presum_kernel(const float *__restrict__ in, float *__restrict__ y,
                                                          const int32_t *__restrict__ pair_row0, const int32_t *__restrict__ yrow_delta,
                                                          int beam0, int nchans, int nyrows, long long nsamps)
{
    const int q = blockIdx.y, b = beam0 + blockIdx.z;
    const int row0 = pair_row0[q], nv = pair_row0[q + 1] - row0;
    const int dlo = yrow_delta[row0];
    const float *x0 = in + ((size_t)b * nchans + 2 * q) * (size_t)nsamps;
    const float *x1 = x0 + nsamps;
    float *o = y + ((size_t)b * nyrows + row0) * (size_t)nsamps;
    const long long t0 = ((long long)blockIdx.x * 256 + threadIdx.x) * 4;
    if (t0 >= nsamps) return;
    float a[4], c[4 + 8];
    const int span = 4 + nv - 1;                       // x1 samples t0 + dlo .. t0 + dlo + span - 1 serve every row (nv <= 9)
#pragma unroll
    for (int i = 0; i < 4; ++i) a[i] = t0 + i < nsamps ? x0[t0 + i] : 0.0f;
#pragma unroll
    for (int i = 0; i < 12; ++i) c[i] = (i < span && t0 + dlo + i < nsamps) ? x1[t0 + dlo + i] : 0.0f;
#pragma unroll
    for (int v = 0; v < 9; ++v) {
        if (v >= nv) break;
        float *ov = o + (size_t)v * nsamps;
        if (t0 + 3 < nsamps) {
            *reinterpret_cast<float4 *>(ov + t0) = make_float4(a[0] + c[v], a[1] + c[v + 1], a[2] + c[v + 2], a[3] + c[v + 3]);
        } else {
#pragma unroll
            for (int i = 0; i < 4; ++i)
                if (t0 + i < nsamps) ov[t0 + i] = a[i] + c[v + i];
        }
    }
}

// the same for the integer path: uint8 in, uint16 sums out (<= 510), so the widening pass is not needed in pair mode
__global__ void __launch_bounds__(256) pair_presum_u8_kernel(const uint8_t *__restrict__ in, uint16_t *__restrict__ y,
                                                             const int32_t *__restrict__ pair_row0, const int32_t *__restrict__ yrow_delta,
                                                             int beam0, int nchans, int nyrows, long long nsamps)
{
    const int q = blockIdx.y, b = beam0 + blockIdx.z;
    const int row0 = pair_row0[q], nv = pair_row0[q + 1] - row0;
    const int dlo = yrow_delta[row0];
    const uint8_t *x0 = in + ((size_t)b * nchans + 2 * q) * (size_t)nsamps;
    const uint8_t *x1 = x0 + nsamps;
    uint16_t *o = y + ((size_t)b * nyrows + row0) * (size_t)nsamps;
    const long long t0 = ((long long)blockIdx.x * 256 + threadIdx.x) * 8;           // nsamps % 8 == 0 on this path
    if (t0 >= nsamps) return;
    unsigned a[8], c[8 + 8];
    const uint2 av = *reinterpret_cast<const uint2 *>(x0 + t0);
#pragma unroll
    for (int i = 0; i < 8; ++i) a[i] = ((i < 4 ? av.x : av.y) >> (8 * (i & 3))) & 0xffu;
    const int span = 8 + nv - 1;
#pragma unroll
    for (int i = 0; i < 16; ++i) c[i] = (i < span && t0 + dlo + i < nsamps) ? x1[t0 + dlo + i] : 0u;
#pragma unroll
    for (int v = 0; v < 9; ++v) {
        if (v >= nv) break;
        uint4 r;
        r.x = (a[0] + c[v]) | ((a[1] + c[v + 1]) << 16);
        r.y = (a[2] + c[v + 2]) | ((a[3] + c[v + 3]) << 16);
        r.z = (a[4] + c[v + 4]) | ((a[5] + c[v + 5]) << 16);
        r.w = (a[6] + c[v + 6]) | ((a[7] + c[v + 7]) << 16);
        *reinterpret_cast<uint4 *>(o + (size_t)v * nsamps + t0) = r;
    }
}

// ------------------------------------------------------------------ host side
struct Geometry {
    int D, T, NW, CS, NOFF;
};
// compiled geometries; index = plan option "tiled_geom_<dtype>"
constexpr Geometry kGeomF32[] = {{4, 28, 11, 16, 12}, {4, 20, 15, 8, 12}, {2, 28, 15, 16, 12}, {4, 28, 12, 16, 12}};   // [2]: coarse DM grids; [3]: 12 warps (setmaxnreg), pair mode only
constexpr Geometry kGeomU16[] = {{2, 40, 15, 16, 12}, {3, 40, 11, 8, 14}, {4, 40, 11, 8, 16}};   // index <= 1: two-phase rows
constexpr int kNumGeomF32 = sizeof(kGeomF32) / sizeof(kGeomF32[0]);
constexpr int kNumGeomU16 = sizeof(kGeomU16) / sizeof(kGeomU16[0]);
constexpr int kPartChansU16 = 256;          // 256 * 255 < 2^16: the most channels a 16-bit lane can take

static inline long long floor_to(long long v, int a) { return v >= 0 ? (v / a) * a : -(((-v) + a - 1) / a) * a; }

// Builds the row-start / per-warp window tables for one geometry.  `al` = samples per 16 bytes of the staged
// element type.  Returns false if this plan's delay spread does not fit the geometry's register window (the
// caller then uses the direct kernel).
static bool build_tables(const mdsm_plan *p, const Geometry &g, int al, bool two_phase, TiledTables &tt, std::vector<int32_t> &h_rs,
                         std::vector<unsigned long long> &h_tab, std::vector<int32_t> &h_sigma)
{
    const int DB = g.D * g.NW, TT = 32 * g.T;
    const int nblk = (p->ndms + DB - 1) / DB;
    const int nslab = (p->nchans + g.CS - 1) / g.CS;
    const int ncp = nslab * g.CS;
    // un-rounded delay increment per DM step at the band edge: the slope the shear splits in half
    const double f_lo = p->f_top + (p->nchans - 1) * p->foff;
    const double smax = 4.148808e3 * p->dm_step * (1.0 / (f_lo * f_lo) - 1.0 / (p->f_top * p->f_top)) / p->tsamp;
    int best_off = 1 << 30;
    double best_shear = 0.0;
    const double cands[] = {0.5, 0.48, 0.52, 0.45, 0.55, 0.4, 0.6, 0.0};
    auto e_of = [&](int blk, int dl, int c, const std::vector<int32_t> &sig) -> long long {
        int d = blk * DB + dl;
        if (d >= p->ndms) d = p->ndms - 1;
        return (long long)p->h_delay[(size_t)d * p->nchans + c] - sig[dl];
    };
    auto make_sigma = [&](double shear, std::vector<int32_t> &sig) {
        sig.resize(DB);
        for (int dl = 0; dl < DB; ++dl) sig[dl] = (int32_t)llround(shear * smax * dl);
    };
    for (double cand : cands) {
        std::vector<int32_t> sig;
        make_sigma(cand, sig);
        int worst = 0;
        for (int blk = 0; blk < nblk && worst < g.NOFF + 8; ++blk)
            for (int w = 0; w < g.NW; ++w)
                for (int c = 0; c < p->nchans; ++c) {
                    long long mn = 1LL << 60, mx = -(1LL << 60);
                    for (int j = 0; j < g.D; ++j) {
                        long long e = e_of(blk, w * g.D + j, c, sig);
                        mn = std::min(mn, e);
                        mx = std::max(mx, e);
                    }
                    worst = std::max(worst, (int)(mx - floor_to(mn, al)));
                }
        if (worst < best_off) { best_off = worst; best_shear = cand; }
    }
    if (best_off >= g.NOFF) return false;
    make_sigma(best_shear, h_sigma);
    h_rs.assign((size_t)nblk * ncp, 0);
    h_tab.assign((size_t)nblk * nslab * g.NW * g.CS, 0ULL);
    // pass 1: row starts and the longest staged row
    long long max_need = 0;
    for (int blk = 0; blk < nblk; ++blk)
        for (int c = 0; c < p->nchans; ++c) {
            long long mn = 1LL << 60;
            for (int dl = 0; dl < DB; ++dl) mn = std::min(mn, e_of(blk, dl, c, h_sigma));
            const long long rs = floor_to(mn, al);
            h_rs[(size_t)blk * ncp + c] = (int32_t)rs;
            for (int w = 0; w < g.NW; ++w) {
                long long wmn = 1LL << 60, wmx = -(1LL << 60);
                for (int j = 0; j < g.D; ++j) {
                    const long long e = e_of(blk, w * g.D + j, c, h_sigma) - rs;
                    wmn = std::min(wmn, e);
                    wmx = std::max(wmx, e);
                }
                const long long A = floor_to(wmn, al);
                const int chunks = (g.T + (int)(wmx - A) + al - 1) / al;
                max_need = std::max(max_need, A + 31LL * g.T + (long long)al * chunks);   // last sample any lane of this warp touches
            }
        }
    const int row_elems = (int)((max_need + al - 1) / al * al);
    const int esize = 16 / al;
    if ((long long)g.CS * row_elems * esize >= (1 << 18)) return false;      // entry holds an 18-bit byte offset
    // pass 2: the per-warp entries (window start includes the row's position in the stage)
    for (int blk = 0; blk < nblk; ++blk)
        for (int c = 0; c < p->nchans; ++c) {
            const long long rs = h_rs[(size_t)blk * ncp + c];
            const int slab = c / g.CS, r = c % g.CS;
            const bool last = (r == g.CS - 1) || (c == p->nchans - 1);
            for (int w = 0; w < g.NW; ++w) {
                long long wmn = 1LL << 60, wmx = -(1LL << 60);
                long long e[8];
                for (int j = 0; j < g.D; ++j) {
                    e[j] = e_of(blk, w * g.D + j, c, h_sigma) - rs;
                    wmn = std::min(wmn, e[j]);
                    wmx = std::max(wmx, e[j]);
                }
                const long long A = floor_to(wmn, al);
                const int chunks = (g.T + (int)(wmx - A) + al - 1) / al;       // 16-byte chunks holding w[0 .. T+maxoff)
                const int extra = chunks - g.T / al;
                unsigned long long lo = (unsigned long long)(((long long)r * row_elems + A) * esize);
                for (int i = 0; i < extra; ++i) lo |= 1ULL << (28 + i);
                if (last) lo |= 1ULL << 31;
                unsigned long long hi = 0;
                for (int j = 0; j < g.D; ++j) {
                    const unsigned long long o = (unsigned long long)(e[j] - A);
                    hi |= (two_phase ? 8 * (o & 1) + (o >> 1) : o) << (8 * j);      // dispatch index of DM j
                }
                h_tab[(((size_t)blk * nslab + slab) * g.NW + w) * g.CS + r] = lo | (hi << 32);
            }
        }
    tt.dms_per_warp = g.D; tt.warps = g.NW; tt.tpt = g.T; tt.cs = g.CS;
    tt.dm_block = DB; tt.n_dm_blocks = nblk; tt.tile_t = TT;
    tt.row_words = row_elems;
    tt.max_off = best_off;
    tt.sigma_max = *std::max_element(h_sigma.begin(), h_sigma.end());
    return true;
}

// Pair mode tables: the rows a DM block stages are (channel pair, delay difference) rows of the pre-summed copy; a row
// is used by the DMs of the block whose delay difference for that pair equals the row's, the others carry offset 15
// (= skip) in the window entry.  Same geometry, shear and entry format as build_tables.
// al = samples per 16 bytes of the staged element; two_phase = dispatch index 8*(o & 1) + (o >> 1) (integer kernel);
// part_pairs > 0: the rows are grouped in parts of that many pairs (16-bit lane capacity), every part of a block padded
// with unused rows to the same number of whole slabs.
static bool build_tables_pairs(const mdsm_plan *p, const Geometry &g, int al, bool two_phase, int part_pairs, TiledTables &tt, std::vector<int32_t> &h_rs,
                               std::vector<unsigned long long> &h_tab, std::vector<int32_t> &h_sigma, std::vector<int32_t> &h_src,
                               std::vector<int32_t> &h_nslab, std::vector<int32_t> &h_ychan, std::vector<int32_t> &h_ydelta)
{
    if (p->nchans % 2 || p->nchans < 2 || g.NOFF > 15) return false;
    const int DB = g.D * g.NW, TT = 32 * g.T, np = p->nchans / 2, esize = 16 / al;
    const int nparts = part_pairs > 0 ? (np + part_pairs - 1) / part_pairs : 1;
    if (part_pairs <= 0) part_pairs = np;
    const int nblk = (p->ndms + DB - 1) / DB;
    auto dly = [&](int d, int c) { return (long long)p->h_delay[(size_t)std::min(d, p->ndms - 1) * p->nchans + c]; };
    // rows of the pre-summed copy: every delay difference a pair takes over the whole DM grid
    std::vector<int> ybase(np), ylo(np);
    h_ychan.clear(); h_ydelta.clear();
    for (int q = 0; q < np; ++q) {
        long long lo = 1LL << 60, hi = -1;
        for (int d = 0; d < p->ndms; ++d) {
            const long long dl = dly(d, 2 * q + 1) - dly(d, 2 * q);
            lo = std::min(lo, dl); hi = std::max(hi, dl);
        }
        if (lo < 0 || hi - lo > 8) return false;                    // the pre-sum kernel holds at most 9 rows of a pair
        ybase[q] = (int)h_ydelta.size(); ylo[q] = (int)lo;
        for (long long dl = lo; dl <= hi; ++dl) h_ydelta.push_back((int32_t)dl);
        h_ychan.push_back(ybase[q]);                                 // first row of pair q (one more entry closes the list)
    }
    h_ychan.push_back((int32_t)h_ydelta.size());
    const double f_lo = p->f_top + (p->nchans - 1) * p->foff;
    const double smax = 4.148808e3 * p->dm_step * (1.0 / (f_lo * f_lo) - 1.0 / (p->f_top * p->f_top)) / p->tsamp;
    h_sigma.resize(DB);
    for (int dl = 0; dl < DB; ++dl) h_sigma[dl] = (int32_t)llround(0.5 * smax * dl);
    // per block: the list of (pair, delta) rows some DM of the block uses
    struct Row { int q, delta; };                 // q < 0: padding row nobody uses
    std::vector<std::vector<Row>> rows(nblk);
    int nslab_max = 0;
    h_nslab.resize(nblk);
    for (int blk = 0; blk < nblk; ++blk) {
        std::vector<std::vector<Row>> part(nparts);
        size_t longest = 0;
        for (int q = 0; q < np; ++q) {
            std::vector<int> seen;
            for (int dl = 0; dl < DB; ++dl) {
                const int d = blk * DB + dl;
                const int de = (int)(dly(d, 2 * q + 1) - dly(d, 2 * q));
                if (std::find(seen.begin(), seen.end(), de) == seen.end()) seen.push_back(de);
            }
            std::sort(seen.begin(), seen.end());
            for (int de : seen) part[q / part_pairs].push_back({q, de});
        }
        for (auto &pr : part) longest = std::max(longest, pr.size());
        const int spp = ((int)longest + g.CS - 1) / g.CS;                  // slabs per part of this block
        for (auto &pr : part) {
            if (nparts > 1) pr.resize((size_t)spp * g.CS, Row{-1, 0});       // a single part may end with a ragged slab
            rows[blk].insert(rows[blk].end(), pr.begin(), pr.end());
        }
        h_nslab[blk] = spp * nparts;
        nslab_max = std::max(nslab_max, h_nslab[blk]);
    }
    const int ncp = nslab_max * g.CS;
    h_rs.assign((size_t)nblk * ncp, 0);
    h_src.assign((size_t)nblk * ncp, -1);
    h_tab.assign((size_t)nblk * nslab_max * g.NW * g.CS, 0ULL);
    auto e_of = [&](int blk, int dl, int c) { return dly(blk * DB + dl, c) - h_sigma[dl]; };
    auto uses = [&](int blk, int dl, const Row &r) { const int d = blk * DB + dl; return r.q >= 0 && dly(d, 2 * r.q + 1) - dly(d, 2 * r.q) == r.delta; };
    long long max_need = 0;
    int worst = 0;
    for (int pass = 0; pass < 2; ++pass) {
        const int row_elems = (int)((max_need + al - 1) / al * al);
        if (pass == 1 && (worst >= g.NOFF || (long long)g.CS * row_elems * esize >= (1 << 18))) return false;
        for (int blk = 0; blk < nblk; ++blk)
            for (int ri = 0; ri < (int)rows[blk].size(); ++ri) {
                const Row &r = rows[blk][ri];
                const int c = r.q >= 0 ? 2 * r.q : 0;
                long long mn = 1LL << 60;
                for (int dl = 0; dl < DB; ++dl)
                    if (uses(blk, dl, r)) mn = std::min(mn, e_of(blk, dl, c));
                const long long rs = r.q >= 0 ? floor_to(mn, al) : 0;
                if (pass == 1 && r.q >= 0) {
                    h_rs[(size_t)blk * ncp + ri] = (int32_t)rs;
                    h_src[(size_t)blk * ncp + ri] = ybase[r.q] + (r.delta - ylo[r.q]);
                }
                const int slab = ri / g.CS, rr = ri % g.CS;
                const bool last = (rr == g.CS - 1) || (ri == (int)rows[blk].size() - 1);
                for (int w = 0; w < g.NW; ++w) {
                    long long wmn = 1LL << 60, wmx = -(1LL << 60), e[8];
                    bool use[8];
                    for (int j = 0; j < g.D; ++j) {
                        use[j] = uses(blk, w * g.D + j, r);
                        e[j] = e_of(blk, w * g.D + j, c) - rs;
                        if (use[j]) { wmn = std::min(wmn, e[j]); wmx = std::max(wmx, e[j]); }
                    }
                    const bool any = wmx >= wmn;
                    const long long A = any ? floor_to(wmn, al) : 0;
                    const int chunks = any ? (g.T + (int)(wmx - A) + al - 1) / al : g.T / al;
                    if (pass == 0) {
                        if (any) {
                            worst = std::max(worst, (int)(wmx - A));
                            max_need = std::max(max_need, A + 31LL * g.T + (long long)al * chunks);
                        }
                        continue;
                    }
                    unsigned long long lo = (unsigned long long)(((long long)rr * row_elems + A) * esize);
                    for (int i = 0; i < chunks - g.T / al; ++i) lo |= 1ULL << (28 + i);
                    if (last) lo |= 1ULL << 31;
                    unsigned long long hi = 0;
                    for (int j = 0; j < g.D; ++j) {
                        const unsigned long long o = (unsigned long long)(e[j] - A);
                        hi |= (use[j] ? (two_phase ? 8 * (o & 1) + (o >> 1) : o) : 0x80ULL) << (8 * j);     // bit 7: skips the row
                    }
                    h_tab[(((size_t)blk * nslab_max + slab) * g.NW + w) * g.CS + rr] = lo | (hi << 32);
                }
            }
        if (pass == 1) {
            tt.row_words = row_elems;
        }
    }
    tt.dms_per_warp = g.D; tt.warps = g.NW; tt.tpt = g.T; tt.cs = g.CS;
    tt.dm_block = DB; tt.n_dm_blocks = nblk; tt.tile_t = TT;
    tt.max_off = worst;
    tt.sigma_max = *std::max_element(h_sigma.begin(), h_sigma.end());
    tt.pairs = true; tt.nslab_max = nslab_max; tt.nyrows = (int)h_ydelta.size(); tt.nparts = nparts;
    return true;
}

template <typename V> static bool upload(V **dptr, const std::vector<V> &h)
{
    if (cudaMalloc((void **)dptr, h.size() * sizeof(V)) != cudaSuccess) return false;
    return cudaMemcpy(*dptr, h.data(), h.size() * sizeof(V), cudaMemcpyHostToDevice) == cudaSuccess;
}

static void free_tables(TiledTables *tt)
{
    cudaFree(tt->d_row_start);
    cudaFree(tt->d_warp_tab);
    cudaFree(tt->d_sigma);
    cudaFree(tt->d_src_row); cudaFree(tt->d_nslab_blk); cudaFree(tt->d_yrow_chan); cudaFree(tt->d_yrow_delta);
    tt->d_row_start = nullptr; tt->d_warp_tab = nullptr; tt->d_sigma = nullptr;
    tt->d_src_row = nullptr; tt->d_nslab_blk = nullptr; tt->d_yrow_chan = nullptr; tt->d_yrow_delta = nullptr;
    tt->pairs = false;
    tt->ok = false;
}

template <typename Tr>
static int launch_tiled(mdsm_plan *p, const TiledTables &tt, const void *d_in, int beam0, int nb, void *d_out, int part_chans,
                        cudaStream_t st)
{
    auto kern = dedisperse_tiled_kernel<Tr>;
    const int nslab = (p->nchans + Tr::CS - 1) / Tr::CS;
    const size_t stage_bytes = (size_t)Tr::CS * tt.row_words * sizeof(typename Tr::In) + (size_t)Tr::NW * Tr::CS * sizeof(unsigned long long);
    int stages = (int)((220 * 1024 - 256) / stage_bytes);
    if (stages > 12) stages = 12;
    MDSM_REQUIRE(stages >= 2, "tiled kernel: staged rows too large for shared memory");
    const size_t smem = stages * stage_bytes + 2 * stages * sizeof(uint64_t) + 16;
    // per launch: the attribute belongs to the current device's copy of the kernel, and the call costs microseconds
    MDSM_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    TiledArgs a;
    a.in = d_in; a.out = d_out;
    a.row_start = tt.d_row_start; a.warp_tab = (const unsigned long long *)tt.d_warp_tab; a.sigma = tt.d_sigma;
    a.src_row = tt.pairs ? tt.d_src_row : nullptr;
    a.nslab_blk = tt.pairs ? tt.d_nslab_blk : nullptr;
    a.nrows_src = tt.pairs ? tt.nyrows : p->nchans;
    a.nparts = tt.pairs ? tt.nparts : 0;
    a.beam0 = beam0; a.nchans = p->nchans; a.nslab = tt.pairs ? tt.nslab_max : nslab; a.ndms = p->ndms;
    a.slabs_per_part = part_chans > 0 ? part_chans / Tr::CS : (tt.pairs ? tt.nslab_max : nslab);
    a.nsamps = p->nsamps; a.nsamps_out = p->nsamps_out;
    a.row_elems = tt.row_words; a.stages = stages;
    a.walk.nblk = tt.n_dm_blocks;
    a.walk.ntile_t = (int)((p->nsamps_out + tt.sigma_max + tt.tile_t - 1) / tt.tile_t);
    a.walk.ntiles = (long long)a.walk.nblk * a.walk.ntile_t * nb;
    const int grid = (int)std::min<long long>(a.walk.ntiles, p->sm_count);
    kern<<<grid, (Tr::NW + Tr::PW) * 32, smem, st>>>(a);
    MDSM_CUDA_TRY(cudaGetLastError());
    p->launches += 1;
    return MDSM_OK;
}

template <int G> using GeomF32 = TraitsF32<kGeomF32[G].D, kGeomF32[G].T, kGeomF32[G].NW, kGeomF32[G].CS, kGeomF32[G].NOFF>;
template <int G> using GeomF32P = TraitsF32P<kGeomF32[G].D, kGeomF32[G].T, kGeomF32[G].NW, kGeomF32[G].CS, kGeomF32[G].NOFF>;
template <int G> using GeomU16 = TraitsU16<kGeomU16[G].D, kGeomU16[G].T, kGeomU16[G].NW, kGeomU16[G].CS, kGeomU16[G].NOFF>;
template <int G> using GeomU16PP = TraitsU16PP<kGeomU16[G].D, kGeomU16[G].T, kGeomU16[G].NW, kGeomU16[G].CS, kGeomU16[G].NOFF>;
template <int G> using GeomU16P = TraitsU16P<kGeomU16[G].D, kGeomU16[G].T, kGeomU16[G].NW, kGeomU16[G].CS, kGeomU16[G].NOFF>;

static int build_one(mdsm_plan *p, const Geometry &g, int al, bool two_phase, int geom, TiledTables &tt)
{
    std::vector<int32_t> rs, sig;
    std::vector<unsigned long long> tab;
    if (!build_tables(p, g, al, two_phase, tt, rs, tab, sig)) return MDSM_OK;
    if (!upload(&tt.d_row_start, rs) || !upload((unsigned long long **)&tt.d_warp_tab, tab) || !upload(&tt.d_sigma, sig)) {
        mdsm_set_error("tiled table upload failed: %s", cudaGetErrorString(cudaGetLastError()));
        return MDSM_ECUDA;
    }
    tt.geom = geom;
    tt.ok = true;
    return MDSM_OK;
}

}  // namespace

int mdsm_tiled_num_geoms(int dtype) { return dtype == MDSM_F32 ? kNumGeomF32 : kNumGeomU16; }

int mdsm_tiled_build_tables(mdsm_plan *p)
{
    free_tables(&p->tiled_f32);
    free_tables(&p->tiled_u8);
    // Rows must be 16-byte aligned for the bulk copies.  tiled_geom_* < 0 = automatic: the first compiled geometry
    // whose register window takes this plan's delay spread (coarser DM grids need fewer DMs per warp).
    if (p->pair_presum && p->nsamps % 4 == 0) {
        std::vector<int32_t> rs, sig, src, nsl, yc, yd;
        std::vector<unsigned long long> tab;
        TiledTables &tt = p->tiled_f32;
        const int pg = p->tiled_geom_f32 == 1 ? 1 : (p->tiled_geom_f32 == 0 ? 0 : 3);   // pair mode is compiled for geometries 0, 1, 3 (default)
        if (build_tables_pairs(p, kGeomF32[pg], 4, false, 0, tt, rs, tab, sig, src, nsl, yc, yd)) {
            if (!upload(&tt.d_row_start, rs) || !upload((unsigned long long **)&tt.d_warp_tab, tab) || !upload(&tt.d_sigma, sig) ||
                !upload(&tt.d_src_row, src) || !upload(&tt.d_nslab_blk, nsl) || !upload(&tt.d_yrow_chan, yc) || !upload(&tt.d_yrow_delta, yd)) {
                mdsm_set_error("tiled table upload failed: %s", cudaGetErrorString(cudaGetLastError()));
                return MDSM_ECUDA;
            }
            tt.geom = pg;
            tt.ok = true;
        }
    }
    if (p->nsamps % 4 == 0 && p->tiled_geom_f32 < kNumGeomF32)
        for (int g = 0; g < 3 && !p->tiled_f32.ok; ++g) {
            if (p->tiled_geom_f32 >= 0 && p->tiled_geom_f32 < 3 && g != p->tiled_geom_f32) continue;
            const int rc = build_one(p, kGeomF32[g], 4, false, g, p->tiled_f32);
            if (rc != MDSM_OK) return rc;
        }
    if (p->pair_presum_u8 && p->nsamps % 8 == 0 && p->tiled_geom_u8 <= 0) {
        std::vector<int32_t> rs, sig, src, nsl, yc, yd;
        std::vector<unsigned long long> tab;
        TiledTables &tt = p->tiled_u8;
        if (build_tables_pairs(p, kGeomU16[0], 8, true, kPartChansU16 / 2, tt, rs, tab, sig, src, nsl, yc, yd)) {
            if (!upload(&tt.d_row_start, rs) || !upload((unsigned long long **)&tt.d_warp_tab, tab) || !upload(&tt.d_sigma, sig) ||
                !upload(&tt.d_src_row, src) || !upload(&tt.d_nslab_blk, nsl) || !upload(&tt.d_yrow_chan, yc) || !upload(&tt.d_yrow_delta, yd)) {
                mdsm_set_error("tiled table upload failed: %s", cudaGetErrorString(cudaGetLastError()));
                return MDSM_ECUDA;
            }
            tt.geom = 0;
            tt.ok = true;
        }
    }
    if (p->nsamps % 8 == 0 && p->tiled_geom_u8 < kNumGeomU16)
        for (int g = 0; g < kNumGeomU16 && !p->tiled_u8.ok; ++g) {
            if (p->tiled_geom_u8 >= 0 && g != p->tiled_geom_u8) continue;
            if (kPartChansU16 % kGeomU16[g].CS != 0) continue;       // parts of 256 channels must be whole slabs
            const int rc = build_one(p, kGeomU16[g], 8, g <= 1, g, p->tiled_u8);
            if (rc != MDSM_OK) return rc;
        }
    return MDSM_OK;
}

void mdsm_tiled_free_tables(mdsm_plan *p)
{
    free_tables(&p->tiled_f32);
    free_tables(&p->tiled_u8);
    cudaFree(p->d_widen);
    p->d_widen = nullptr;
    p->widen_bytes = 0;
    cudaFree(p->d_pairs);
    p->d_pairs = nullptr;
    p->pairs_bytes = 0;
}

int mdsm_launch_dedisperse_tiled(mdsm_plan *p, const void *d_in, int dtype, int beam0, int nb, void *d_out,
                                 cudaStream_t st)
{
    if (dtype == MDSM_F32) {
        const TiledTables &tt = p->tiled_f32;
        if (tt.pairs) {
            // pre-sum the channel pairs of these beams into the plan's scratch (allocated on first use), then walk its rows
            const size_t need = (size_t)p->nbeams * tt.nyrows * (size_t)p->nsamps * sizeof(float);
            if (p->pairs_bytes < need) {
                cudaFree(p->d_pairs);
                p->d_pairs = nullptr;
                p->pairs_bytes = 0;
                if (cudaMalloc(&p->d_pairs, need) != cudaSuccess) {
                    // no room for the pre-summed copy: this plan goes on without pair pre-sums (tables rebuilt once;
                    // the caller's stream may still run kernels of this plan, so wait for them before freeing tables)
                    (void)cudaGetLastError();
                    p->d_pairs = nullptr;
                    p->pair_presum = 0;
                    MDSM_CUDA_TRY(cudaDeviceSynchronize());
                    const int rc = mdsm_tiled_build_tables(p);
                    if (rc != MDSM_OK) return rc;
                    if (!p->tiled_f32.ok) return mdsm_launch_dedisperse_direct(p, d_in, dtype, beam0, nb, d_out, st);
                    return mdsm_launch_dedisperse_tiled(p, d_in, dtype, beam0, nb, d_out, st);
                }
                p->pairs_bytes = need;
            }
            dim3 grid((unsigned)((p->nsamps / 4 + 255) / 256), p->nchans / 2, nb);
            MDSM_REQUIRE(p->nchans / 2 <= 65535 && nb <= 65535, "pair pre-sum: grid too large");
            pair_presum_kernel<<<grid, 256, 0, st>>>((const float *)d_in, (float *)p->d_pairs, tt.d_yrow_chan, tt.d_yrow_delta, beam0,
                                                     p->nchans, tt.nyrows, p->nsamps);
            MDSM_CUDA_TRY(cudaGetLastError());
            p->launches += 1;
            if (tt.geom == 1) return launch_tiled<GeomF32P<1>>(p, tt, p->d_pairs, beam0, nb, d_out, 0, st);
            if (tt.geom == 3) return launch_tiled<GeomF32P<3>>(p, tt, p->d_pairs, beam0, nb, d_out, 0, st);
            return launch_tiled<GeomF32P<0>>(p, tt, p->d_pairs, beam0, nb, d_out, 0, st);
        }
        switch (tt.geom) {
            case 0: return launch_tiled<GeomF32<0>>(p, tt, d_in, beam0, nb, d_out, 0, st);
            case 1: return launch_tiled<GeomF32<1>>(p, tt, d_in, beam0, nb, d_out, 0, st);
            case 2: return launch_tiled<GeomF32<2>>(p, tt, d_in, beam0, nb, d_out, 0, st);
        }
        mdsm_set_error("tiled kernel: bad geometry index %d", tt.geom);
        return MDSM_EINVAL;
    }
    // uint8: widen the beams of this call to uint16 in the plan's scratch (allocated on first use, whole plan)
    const TiledTables &tt = p->tiled_u8;
    const size_t beam_elems = (size_t)p->nchans * (size_t)p->nsamps;
    if (tt.pairs) {
        // pair mode: the pre-pass writes uint16 pair sums (which also widens), the tiled kernel walks its rows
        const size_t needp = (size_t)p->nbeams * tt.nyrows * (size_t)p->nsamps * sizeof(uint16_t);
        if (p->widen_bytes < needp) {
            cudaFree(p->d_widen);
            p->d_widen = nullptr;
            p->widen_bytes = 0;
            if (cudaMalloc(&p->d_widen, needp) != cudaSuccess) {
                (void)cudaGetLastError();
                p->d_widen = nullptr;
                p->pair_presum_u8 = 0;                       // no room: go on without pair pre-sums (see the fp32 path)
                MDSM_CUDA_TRY(cudaDeviceSynchronize());
                const int rc = mdsm_tiled_build_tables(p);
                if (rc != MDSM_OK) return rc;
                if (!p->tiled_u8.ok) return mdsm_launch_dedisperse_direct(p, d_in, dtype, beam0, nb, d_out, st);
                return mdsm_launch_dedisperse_tiled(p, d_in, dtype, beam0, nb, d_out, st);
            }
            p->widen_bytes = needp;
        }
        dim3 grid((unsigned)((p->nsamps / 8 + 255) / 256), p->nchans / 2, nb);
        MDSM_REQUIRE(p->nchans / 2 <= 65535 && nb <= 65535, "pair pre-sum: grid too large");
        pair_presum_u8_kernel<<<grid, 256, 0, st>>>((const uint8_t *)d_in, (uint16_t *)p->d_widen, tt.d_yrow_chan, tt.d_yrow_delta, beam0,
                                                    p->nchans, tt.nyrows, p->nsamps);
        MDSM_CUDA_TRY(cudaGetLastError());
        p->launches += 1;
        return launch_tiled<GeomU16PP<0>>(p, tt, p->d_widen, beam0, nb, d_out, 0, st);
    }
    const size_t need = (size_t)p->nbeams * beam_elems * sizeof(uint16_t);
    if (p->widen_bytes < need) {
        cudaFree(p->d_widen);
        p->d_widen = nullptr;
        p->widen_bytes = 0;
        MDSM_CUDA_TRY(cudaMalloc(&p->d_widen, need));
        p->widen_bytes = need;
    }
    const uint8_t *src = (const uint8_t *)d_in + (size_t)beam0 * beam_elems;
    uint16_t *dst = (uint16_t *)p->d_widen + (size_t)beam0 * beam_elems;
    const size_t n8 = (size_t)nb * beam_elems / 8;
    widen_u8_kernel<<<p->sm_count * 8, 256, 0, st>>>((const uint2 *)src, (uint4 *)dst, n8);
    MDSM_CUDA_TRY(cudaGetLastError());
    p->launches += 1;
    switch (tt.geom) {
        case 0: return launch_tiled<GeomU16P<0>>(p, tt, p->d_widen, beam0, nb, d_out, kPartChansU16, st);
        case 1: return launch_tiled<GeomU16P<1>>(p, tt, p->d_widen, beam0, nb, d_out, kPartChansU16, st);
        case 2: return launch_tiled<GeomU16<2>>(p, tt, p->d_widen, beam0, nb, d_out, kPartChansU16, st);
    }
    mdsm_set_error("tiled kernel: bad geometry index %d", tt.geom);
    return MDSM_EINVAL;
}
