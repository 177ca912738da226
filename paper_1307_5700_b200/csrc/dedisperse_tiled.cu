// Tiled brute-force dedispersion for sm_100a (BASELINE.json north_star item 2).
//
//   out[b][d][t] = sum_c in[b][c][t + delay(d,c)]
//
// Work decomposition:
//   CTA   = one beam x one block of DB = NW*D consecutive DM trials x one time tile of 32*T samples.
//   warp  = D consecutive DM trials of the block, all 32*T samples of the tile.
//   thread= D x T accumulators in registers: T CONSECUTIVE samples (lane*T ...) of each of its D DMs.
// Per channel a thread loads ONE register window of T + (spread of its D delays) consecutive samples
// from shared memory with conflict-free 128-bit loads (T/4 is odd) and adds it, at D different
// register offsets, into its D accumulator rows -- every shared-memory word feeds ~3 adds, which is
// what lifts the kernel off the 32 words/clk/SM shared-memory ceiling (25 % of the add peak).
// The offsets are warp-uniform; they select straight-line add blocks through a threaded chain of
// indirect branches (chain_gen.h).  fp32 accumulators and window are packed f32x2 register pairs so
// that an even offset costs T/2 issue slots (FADD2) -- the FMA pipe, not the issue port, is the limit.
// The time axis is SHEARED: DM d of a block owns outputs [tile_t0 - sigma_d, tile_t0 - sigma_d + 32T)
// with sigma_d ~ half the band-edge delay slope, which halves the spread of the D windows (and of
// the staged rows) compared with an unsheared tile.
// Staging: a producer warp streams channel slabs (CS rows of `row_words` samples, each starting at
// its own 16-byte-aligned delay-dependent offset) into a ring of shared-memory stages with 1-D TMA
// bulk copies (cp.async.bulk ... mbarrier::complete_tx), full/empty mbarriers per stage.
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
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "W: mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra D;\n\t"
        "bra W;\n\t"
        "D:\n\t"
        "}" ::"r"(smem_u32(bar)), "r"(parity)
        : "memory");
}
// producer-side wait: the producer runs several stages ahead, so it sleeps between polls instead of
// spinning (a spinning producer warp took 12 % of the SM's issue slots in the r1b profile)
__device__ __forceinline__ void mbar_wait_sleep(uint64_t *bar, uint32_t parity)
{
    uint32_t done;
    for (;;) {
        asm volatile(
            "{\n\t"
            ".reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t"
            "}" : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
        if (done) break;
        __nanosleep(256);
    }
}
__device__ __forceinline__ void bulk_g2s(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void lds128(unsigned long long &a, unsigned long long &b, uint32_t addr)
{
    asm volatile("ld.shared.v2.b64 {%0, %1}, [%2];" : "=l"(a), "=l"(b) : "r"(addr));
}

// predicated form: one SASS instruction, no branch (the registers keep stale data when pred is false)
__device__ __forceinline__ void lds128_if(unsigned long long &a, unsigned long long &b, uint32_t addr, bool pred)
{
    asm volatile("{ .reg .pred q; setp.ne.u32 q, %3, 0; @q ld.shared.v2.b64 {%0, %1}, [%2]; }" : "=l"(a), "=l"(b) : "r"(addr), "r"((unsigned)pred));
}

// Stores v[0..T) to orow[ts .. ts+T), clipped to [0, n).  Rows are 16-byte aligned; ts is not (the
// shear is a whole number of samples), so the head up to the next multiple of 4 goes out as scalars and
// the rest as 128-bit stores.  The head length is warp-uniform: one switch, static register indexing.
template <int T, int H, typename V>
__device__ __forceinline__ void store_row_h(V *orow, long long ts, long long n, const V (&v)[T])
{
#pragma unroll
    for (int i = 0; i < H; ++i)
        if (ts + i >= 0 && ts + i < n) orow[ts + i] = v[i];
#pragma unroll
    for (int i = H; i + 3 < T; i += 4) {
        const long long t = ts + i;
        if (t >= 0 && t + 3 < n) {
            uint4 q;
            q.x = reinterpret_cast<const uint32_t &>(v[i]); q.y = reinterpret_cast<const uint32_t &>(v[i + 1]);
            q.z = reinterpret_cast<const uint32_t &>(v[i + 2]); q.w = reinterpret_cast<const uint32_t &>(v[i + 3]);
            *reinterpret_cast<uint4 *>(orow + t) = q;
        } else {
#pragma unroll
            for (int k = 0; k < 4; ++k)
                if (t + k >= 0 && t + k < n) orow[t + k] = v[i + k];
        }
    }
#pragma unroll
    for (int i = H + (T - H) / 4 * 4; i < T; ++i)
        if (ts + i >= 0 && ts + i < n) orow[ts + i] = v[i];
}
template <int T, typename V>
__device__ __forceinline__ void store_row(V *orow, long long ts, long long n, const V (&v)[T])
{
    static_assert(sizeof(V) == 4, "32-bit outputs");
    switch ((int)((4 - (ts & 3)) & 3)) {
        case 0: store_row_h<T, 0>(orow, ts, n, v); break;
        case 1: store_row_h<T, 1>(orow, ts, n, v); break;
        case 2: store_row_h<T, 2>(orow, ts, n, v); break;
        default: store_row_h<T, 3>(orow, ts, n, v); break;
    }
}

// ------------------------------------------------------------------ producer (shared by the dtypes)
// Lane r < CS copies row r of every slab, lane CS copies the slab's slice of the warp table.
template <typename TIn, int NW, int CS>
__device__ __forceinline__ void producer_loop(const TIn *__restrict__ beam_in, const int32_t *__restrict__ rs,
                                              const unsigned long long *__restrict__ wtab, unsigned char *rows,
                                              unsigned long long *tabs, uint64_t *full, uint64_t *empty, long long tile_t0,
                                              int nchans, int nslab, long long nsamps, int row_elems, int stages, int lane)
{
    int st = 0;
    uint32_t ph = 1;            // parity of the empty-barrier phase to wait for (first lap: no wait)
    for (int slab = 0; slab < nslab; ++slab, ++st) {
        if (st == stages) { st = 0; ph ^= 1; }
        if (slab >= stages) mbar_wait_sleep(&empty[st], ph);
        if (lane < CS) {
            const int c = slab * CS + lane;
            uint32_t bytes = 0;
            long long lo = 0, g0 = 0;
            if (c < nchans) {
                g0 = tile_t0 + rs[c];
                lo = g0 < 0 ? 0 : g0;
                long long hi = g0 + row_elems;
                if (hi > nsamps) hi = nsamps;
                if (hi > lo) bytes = (uint32_t)((hi - lo) * sizeof(TIn));
            }
            mbar_arrive_expect_tx(&full[st], bytes);
            if (bytes)
                bulk_g2s(rows + (((size_t)st * CS + lane) * row_elems + (lo - g0)) * sizeof(TIn),
                         beam_in + (size_t)c * nsamps + lo, bytes, &full[st]);
        } else if (lane == CS) {
            const uint32_t bytes = NW * CS * sizeof(unsigned long long);
            mbar_arrive_expect_tx(&full[st], bytes);
            bulk_g2s(tabs + (size_t)st * NW * CS, wtab + (size_t)slab * NW * CS, bytes, &full[st]);
        }
    }
}

// ------------------------------------------------------------------ fp32 kernel
// warp_tab entry (64 bit): bits 0..15 window start in 16-byte units relative to the stage base (row r
// included), bits 16..19 number of 16-byte chunks to load beyond T/4 (adaptive window), byte 3+j:
// register offset of DM j.
template <int D, int T, int NW, int CS, int NOFF>
__global__ void __launch_bounds__((NW + 1) * 32, 1)
dedisperse_tiled_f32_kernel(const float *__restrict__ in, float *__restrict__ out, const int32_t *__restrict__ row_start,
                            const unsigned long long *__restrict__ warp_tab, const int32_t *__restrict__ sigma, int beam0,
                            int nchans, int nslab, int ndms, long long nsamps, long long nsamps_out, int row_words,
                            int stages)
{
    static_assert(T % 4 == 0 && (T / 4) % 2 == 1, "T/4 must be odd (bank-conflict-free 128-bit window loads)");
    static_assert(D <= 5, "table entry holds at most 5 offsets");
    using Chain = ChainF32<D, T, NOFF>;
    constexpr int W2 = Chain::W2;           // window length in f32x2 pairs
    constexpr int DB = D * NW;
    extern __shared__ __align__(128) unsigned char smem[];
    const size_t stage_bytes = (size_t)CS * row_words * sizeof(float);
    unsigned long long *tabs = reinterpret_cast<unsigned long long *>(smem + (size_t)stages * stage_bytes);
    uint64_t *full = reinterpret_cast<uint64_t *>(tabs + (size_t)stages * NW * CS);
    uint64_t *empty = full + stages;

    const int blk = blockIdx.x;
    const long long tile_t0 = (long long)blockIdx.y * (32 * T);
    const int b = beam0 + blockIdx.z;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    if (threadIdx.x == 0) {
        for (int s = 0; s < stages; ++s) {
            mbar_init(&full[s], CS + 1);
            mbar_init(&empty[s], NW);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp == NW) {
        if (lane <= CS)
            producer_loop<float, NW, CS>(in + (size_t)b * nchans * (size_t)nsamps, row_start + (size_t)blk * nslab * CS,
                                         warp_tab + (size_t)blk * nslab * NW * CS, smem, tabs, full, empty, tile_t0, nchans,
                                         nslab, nsamps, row_words, stages, lane);
        return;
    }

    // ===== consumer warps =====
    unsigned long long acc[D][T / 2];
#pragma unroll
    for (int j = 0; j < D; ++j)
#pragma unroll
        for (int i = 0; i < T / 2; ++i) acc[j][i] = 0ull;      // (+0.f, +0.f)

    const uint32_t lane_base = smem_u32(smem) + lane * (T * 4);
    int st = 0;
    uint32_t ph = 0;
#pragma unroll 1
    for (int slab = 0; slab < nslab; ++slab, ++st) {
        if (st == stages) { st = 0; ph ^= 1; }
        mbar_wait(&full[st], ph);
        const unsigned long long *tab = tabs + ((size_t)st * NW + warp) * CS;
        const uint32_t sbase = lane_base + (uint32_t)(st * stage_bytes);
        const int nc = min(CS, nchans - slab * CS);
        unsigned long long wt = tab[0];
#pragma unroll 1
        for (int r = 0; r < nc; ++r) {
            const unsigned lo32 = (unsigned)wt, hi32 = (unsigned)(wt >> 32);
            wt = tab[r + 1];                                  // prefetch (the entry after the last one is never used)
            const uint32_t p = sbase + ((lo32 & 0xffffu) << 4);
            const int extra = (lo32 >> 16) & 0xf;
            unsigned long long w[W2];
#pragma unroll
            for (int i = 0; i < T / 4; ++i) lds128(w[2 * i], w[2 * i + 1], p + 16 * i);
#pragma unroll
            for (int i = T / 4; i < W2 / 2; ++i) lds128_if(w[2 * i], w[2 * i + 1], p + 16 * i, i - T / 4 < extra);
            Chain::run(acc, w, lo32, hi32);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[st]);
    }

    // ===== epilogue: each thread owns T consecutive outputs of each of its D DMs =====
#pragma unroll
    for (int j = 0; j < D; ++j) {
        const int dl = warp * D + j;
        const int d = blk * DB + dl;
        if (d >= ndms) continue;
        float v[T];
#pragma unroll
        for (int i = 0; i < T / 2; ++i) {
            v[2 * i] = __uint_as_float((unsigned)acc[j][i]);
            v[2 * i + 1] = __uint_as_float((unsigned)(acc[j][i] >> 32));
        }
        const long long ts = tile_t0 - sigma[dl] + (long long)lane * T;
        store_row<T>(out + ((size_t)b * ndms + d) * (size_t)nsamps, ts, nsamps_out, v);
    }
}

// ------------------------------------------------------------------ host side
struct Geometry {
    int D, T, NW, CS, NOFF;
};
// compiled fp32 geometries; index = plan option "tiled_geom"
constexpr Geometry kGeomF32[] = {{4, 28, 11, 8, 12}, {4, 20, 15, 8, 12}, {5, 20, 11, 8, 16}, {4, 28, 11, 8, 16}};
constexpr int kNumGeomF32 = sizeof(kGeomF32) / sizeof(kGeomF32[0]);

static inline long long floor4(long long v) { return v >= 0 ? (v / 4) * 4 : -(((-v) + 3) / 4) * 4; }

// Builds the row-start / per-warp window tables for one geometry.  Returns false if this plan's
// delay spread does not fit the geometry's register window (the caller then uses the direct kernel).
static bool build_tables(const mdsm_plan *p, const Geometry &g, TiledTables &tt, std::vector<int32_t> &h_rs,
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
                    worst = std::max(worst, (int)(mx - floor4(mn)));
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
            const long long rs = floor4(mn);
            h_rs[(size_t)blk * ncp + c] = (int32_t)rs;
            for (int w = 0; w < g.NW; ++w) {
                long long wmn = 1LL << 60, wmx = -(1LL << 60);
                for (int j = 0; j < g.D; ++j) {
                    const long long e = e_of(blk, w * g.D + j, c, h_sigma) - rs;
                    wmn = std::min(wmn, e);
                    wmx = std::max(wmx, e);
                }
                const long long A = floor4(wmn);
                const int chunks = (g.T + (int)(wmx - A) + 3) / 4;
                max_need = std::max(max_need, A + 31LL * g.T + 4LL * chunks);   // last word any lane of this warp touches
            }
        }
    const int row_words = (int)((max_need + 3) / 4 * 4);
    if ((long long)g.CS * row_words / 4 > 0xffff) return false;
    // pass 2: the per-warp entries (window start includes the row's position in the stage)
    for (int blk = 0; blk < nblk; ++blk)
        for (int c = 0; c < p->nchans; ++c) {
            const long long rs = h_rs[(size_t)blk * ncp + c];
            const int slab = c / g.CS, r = c % g.CS;
            for (int w = 0; w < g.NW; ++w) {
                long long wmn = 1LL << 60, wmx = -(1LL << 60);
                long long e[8];
                for (int j = 0; j < g.D; ++j) {
                    e[j] = e_of(blk, w * g.D + j, c, h_sigma) - rs;
                    wmn = std::min(wmn, e[j]);
                    wmx = std::max(wmx, e[j]);
                }
                const long long A = floor4(wmn);
                const int chunks = (g.T + (int)(wmx - A) + 3) / 4;       // 16-byte chunks holding w[0 .. T+maxoff)
                const int extra = chunks - g.T / 4;
                unsigned long long ent = (unsigned long long)((long long)r * row_words / 4 + A / 4) | ((unsigned long long)extra << 16);
                for (int j = 0; j < g.D; ++j) ent |= (unsigned long long)(e[j] - A) << (24 + 8 * j);
                h_tab[(((size_t)blk * nslab + slab) * g.NW + w) * g.CS + r] = ent;
            }
        }
    tt.dms_per_warp = g.D; tt.warps = g.NW; tt.tpt = g.T;
    tt.dm_block = DB; tt.n_dm_blocks = nblk; tt.tile_t = TT;
    tt.row_words = row_words;
    tt.max_off = best_off;
    tt.sigma_max = *std::max_element(h_sigma.begin(), h_sigma.end());
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
    tt->d_row_start = nullptr; tt->d_warp_tab = nullptr; tt->d_sigma = nullptr;
    tt->ok = false;
}

template <int G>
static int launch_f32(mdsm_plan *p, const TiledTables &tt, const float *d_in, int beam0, int nb, float *d_out, cudaStream_t st)
{
    constexpr Geometry g = kGeomF32[G];
    auto kern = dedisperse_tiled_f32_kernel<g.D, g.T, g.NW, g.CS, g.NOFF>;
    const int nslab = (p->nchans + g.CS - 1) / g.CS;
    const size_t stage_bytes = (size_t)g.CS * tt.row_words * sizeof(float) + (size_t)g.NW * g.CS * sizeof(unsigned long long);
    int stages = (int)((220 * 1024 - 256) / stage_bytes);
    if (stages > 8) stages = 8;
    if (stages > nslab) stages = nslab;
    MDSM_REQUIRE(stages >= 2 || nslab == 1, "tiled kernel: staged rows too large for shared memory");
    const size_t smem = stages * stage_bytes + 2 * stages * sizeof(uint64_t) + 16;
    static thread_local size_t smem_set = 0;
    if (smem > smem_set) {
        MDSM_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        smem_set = smem;
    }
    const long long ntile = (p->nsamps_out + tt.sigma_max + tt.tile_t - 1) / tt.tile_t;
    MDSM_REQUIRE(ntile <= 65535 && nb <= 65535, "tiled kernel: grid too large");
    dim3 grid(tt.n_dm_blocks, (unsigned)ntile, nb);
    kern<<<grid, (g.NW + 1) * 32, smem, st>>>(d_in, d_out, tt.d_row_start, (const unsigned long long *)tt.d_warp_tab, tt.d_sigma,
                                              beam0, p->nchans, nslab, p->ndms, p->nsamps, p->nsamps_out, tt.row_words, stages);
    MDSM_CUDA_TRY(cudaGetLastError());
    p->launches += 1;
    return MDSM_OK;
}

}  // namespace

int mdsm_tiled_num_geoms(int dtype) { return dtype == MDSM_F32 ? kNumGeomF32 : 0; }

int mdsm_tiled_build_tables(mdsm_plan *p)
{
    free_tables(&p->tiled_f32);
    free_tables(&p->tiled_u8);
    if (p->nsamps % 4 != 0) return MDSM_OK;   // rows must be 16-byte aligned for the bulk copies
    std::vector<int32_t> rs, sig;
    std::vector<unsigned long long> tab;
    TiledTables &tt = p->tiled_f32;
    if (p->tiled_geom_f32 < 0 || p->tiled_geom_f32 >= kNumGeomF32) return MDSM_OK;
    if (!build_tables(p, kGeomF32[p->tiled_geom_f32], tt, rs, tab, sig)) return MDSM_OK;
    if (!upload(&tt.d_row_start, rs) || !upload((unsigned long long **)&tt.d_warp_tab, tab) || !upload(&tt.d_sigma, sig)) {
        mdsm_set_error("tiled table upload failed: %s", cudaGetErrorString(cudaGetLastError()));
        return MDSM_ECUDA;
    }
    tt.geom = p->tiled_geom_f32;
    tt.ok = true;
    return MDSM_OK;
}

void mdsm_tiled_free_tables(mdsm_plan *p)
{
    free_tables(&p->tiled_f32);
    free_tables(&p->tiled_u8);
}

int mdsm_launch_dedisperse_tiled(mdsm_plan *p, const void *d_in, int dtype, int beam0, int nb, void *d_out,
                                 cudaStream_t st)
{
    MDSM_REQUIRE(dtype == MDSM_F32, "tiled kernel: only MDSM_F32 so far");
    const TiledTables &tt = p->tiled_f32;
    const float *in = (const float *)d_in;
    float *out = (float *)d_out;
    switch (tt.geom) {
        case 0: return launch_f32<0>(p, tt, in, beam0, nb, out, st);
        case 1: return launch_f32<1>(p, tt, in, beam0, nb, out, st);
        case 2: return launch_f32<2>(p, tt, in, beam0, nb, out, st);
        case 3: return launch_f32<3>(p, tt, in, beam0, nb, out, st);
    }
    mdsm_set_error("tiled kernel: bad geometry index %d", tt.geom);
    return MDSM_EINVAL;
}
