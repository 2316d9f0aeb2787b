// mask_decode.cu — chorus_mask_to_index and chorus_visit_refresh kernels (HBM-bound integer work).
//
// Decode (PAPER.md:L81/L87/L93; include/chorus.h): packed block bitmask [rows][words] ->
// CSR (row_ptr, col_idx), ascending inside each row.  ONE pass over the bitmask, one launch (plus a
// memset of the small look-back array): the bitmask is taken as a flat array of rows*words words,
// cut into tiles of 256*WPT words, WPT consecutive words per thread; a block
//   1. loads its tile, clears the pad bits of the last word of each row and counts;
//   2. scans the counts inside the block and gets the number of set bits in front of its tile with
//      a decoupled look-back over the per-tile status words, 256 at a time (tiles are taken in
//      ticket order, so a tile only ever waits for tiles that already run);
//   3. writes row_ptr for every row that begins in the tile; the set bits of the tile's words are walked into a
//      shared-memory staging buffer (before the look-back when the whole tile fits) - in the plain geometry after
//      a counting sort of the words by popcount, so that the lanes of a warp walk equally long words - which the
//      block copies to col_idx in contiguous, coalesced runs.  Entries that fit 16 bits are staged in 16-bit
//      slots (24 KB instead of 44 KB of shared memory: eight resident blocks per SM instead of five).
// Algorithmic traffic: 4*(rows*words) read + 4*(rows+1) + 4*nnz written; nothing is read twice.
#include <algorithm>
#include <mutex>

#include "chorus_internal.h"

namespace chorus {
namespace {

constexpr int DEC_THREADS = 256;
constexpr int DEC_WARPS = DEC_THREADS / 32;
constexpr int DEC_BLOCKS16 = 8;                                  // resident blocks per SM aimed at with 16-bit slots (32 registers)
// col_idx entries staged per round: 44 KB of 32-bit or 24 KB of 16-bit slots (entries that fit 16 bits are staged
// in 16 bits: more resident blocks per SM)
template <typename StageT>
constexpr int stage_entries() { return sizeof(StageT) == 2 ? 12288 : 11264; }

// Staging-buffer slot of entry e: the low five bits are XORed with the next five, so that threads whose runs
// start 8, 16 or 32 entries apart (25 %, 50 %, full density) hit different banks when they all write their
// k-th entry, while 32 consecutive entries still fall into 32 different banks for the copy-out.
__device__ __forceinline__ int slot(int e) { return e ^ ((e >> 5) & 31); }

// The set bits of x, ascending, into the staging buffer from entry e on.  Walked from the top bit down into
// descending slots: the position of the highest set bit is ONE instruction (FLO), where the lowest one costs a
// bit reversal as well.  val(b) gives the entry of bit b.
template <typename StageT, typename F>
__device__ __forceinline__ void walk_word(uint32_t x, int e, StageT* s_stage, F val) {
    int pos = e + __popc(x) - 1;
    while (x) {
        int b;
        asm("bfind.u32 %0, %1;" : "=r"(b) : "r"(x));   // one FLO; `31 - __clz(x)` compiles to a clz and its way back
        x ^= 1u << b;
        s_stage[slot(pos)] = static_cast<StageT>(val(b));
        --pos;
    }
}

// per-tile status word: bits 63..62 = state (0 empty, 1 aggregate of the tile, 2 inclusive prefix),
// low 32 bits = value.  Written and read with single 64-bit relaxed accesses.
constexpr unsigned long long ST_AGG = 1ull << 62, ST_INC = 2ull << 62;

__device__ __forceinline__ void st_status(unsigned long long* p, unsigned long long v) {
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ unsigned long long ld_status(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}

// Source of the words when the mask is stored in the paper's 64 x 128 geometry (include/chorus.h,
// chorus_mask_to_index_64x128): the tile mask of a 128-row block is never materialised.  Word wr of row r
// (l, h, qb) = the union of mask rows 2 qb and 2 qb + 1, key blocks 16 wr .. 16 wr + 15, each spread over its two
// 64-key tiles; fu / fl keep the 16 source bits of the upper / lower mask row for the per-half flags.
struct GeoSrc {
    const uint32_t* bm64;
    int nq64, nq128, nk128, words128;
};
__device__ __forceinline__ uint32_t spread16(uint32_t x) {      // bit b of the low 16 -> bits 2b, 2b+1
    x = (x | (x << 8)) & 0x00ff00ffu;
    x = (x | (x << 4)) & 0x0f0f0f0fu;
    x = (x | (x << 2)) & 0x33333333u;
    x = (x | (x << 1)) & 0x55555555u;
    return x | (x << 1);
}
__device__ __forceinline__ uint32_t geo_word(const GeoSrc& g, uint32_t r, int wr, uint32_t& fu, uint32_t& fl) {
    const uint32_t hd = r / static_cast<uint32_t>(g.nq128), qb = r - hd * static_cast<uint32_t>(g.nq128);
    const uint32_t* up = g.bm64 + (static_cast<int64_t>(hd) * g.nq64 + 2 * qb) * g.words128;
    const int wi = wr >> 1, sh = 16 * (wr & 1);
    uint32_t a = __ldg(up + wi);
    uint32_t b = (2 * qb + 1 < static_cast<uint32_t>(g.nq64)) ? __ldg(up + g.words128 + wi) : 0u;
    const int rem = g.nk128 - wi * 32;                          // valid key blocks of this source word
    if (rem < 32) {
        const uint32_t m = (1u << rem) - 1u;
        a &= m;
        b &= m;
    }
    fu = (a >> sh) & 0xffffu;
    fl = (b >> sh) & 0xffffu;
    return spread16(fu | fl);
}
// entry of tile bit b (tile index t): t | upper half does not keep it << 30 | lower half does not << 31
__device__ __forceinline__ int32_t geo_entry(int t, int b, uint32_t fu, uint32_t fl) {
    const uint32_t nu = (~fu >> (b >> 1)) & 1u, nl = (~fl >> (b >> 1)) & 1u;
    return static_cast<int32_t>(static_cast<uint32_t>(t) | (nu << 30) | (nl << 31));
}

// A staged entry on its way out: 32-bit as it is; 16-bit with the two per-half flags of the
// 64 x 128 geometry moved from bits 30 / 31 to bits 14 / 15.
template <typename IdxT, bool kGeo>
__device__ __forceinline__ IdxT out_entry(int32_t e) {
    if constexpr (sizeof(IdxT) == 4) return static_cast<IdxT>(e);
    const uint32_t u = static_cast<uint32_t>(e);
    if constexpr (kGeo) return static_cast<IdxT>((u & 0x3fffu) | ((u >> 30) << 14));
    return static_cast<IdxT>(u);
}
// the same on the way INTO the staging buffer (StageT 16-bit: the conversion happens here) and out of it
template <typename StageT, bool kGeo>
__device__ __forceinline__ StageT stage_entry(int32_t e) { return out_entry<StageT, kGeo>(e); }
template <typename IdxT, typename StageT, bool kGeo>
__device__ __forceinline__ IdxT unstage_entry(StageT v) {
    if constexpr (sizeof(StageT) == 2) return static_cast<IdxT>(v);     // already in its final form (zero-extended)
    else return out_entry<IdxT, kGeo>(static_cast<int32_t>(v));
}

// WPT consecutive words per thread: 4 for large mask sets (fewer scans, divisions and status words per
// word), 1 for a single layer (more, smaller tiles: one 480p layer is only 160 K words)
template <int WPT, bool kGeo, typename IdxT, typename StageT>
__global__ void __launch_bounds__(DEC_THREADS, sizeof(StageT) == 2 ? DEC_BLOCKS16 : 5)
decode_tiles_kernel(const uint32_t* __restrict__ bitmask, int64_t rows, int nk, int words,
                    int32_t* __restrict__ row_ptr, IdxT* __restrict__ col_idx, int64_t col_cap,
                    unsigned long long* __restrict__ status /* [0] = ticket counter, [1 + t] = tile t */,
                    const GeoSrc geo) {
    static_assert(sizeof(StageT) == 4 || sizeof(IdxT) == 2 || !kGeo, "flagged 32-bit entries need 32-bit slots");
    constexpr int STAGE = stage_entries<StageT>();
    __shared__ __align__(16) unsigned char s_raw[STAGE * sizeof(StageT)];
    StageT* s_stage = reinterpret_cast<StageT*>(s_raw);          // entry e at slot(e)
    __shared__ int s_warp[DEC_WARPS];
    __shared__ int2 s_look[DEC_WARPS];
    __shared__ int s_tile, s_base;
    constexpr int TILE_WORDS = DEC_THREADS * WPT;
    // words of the tile in descending order of their popcount (see "balanced walk" below): the word and
    // (staging offset | word-in-row << 14); s_bkt: per popcount 32..1 a counter, then the bucket's first position
    // They live in the tail of the staging buffer, which such a tile does not reach.
    constexpr bool kSort = !kGeo;
    constexpr int SORT_MAX = STAGE - 2 * TILE_WORDS * 4 / static_cast<int>(sizeof(StageT));   // most entries of a tile walked sorted
    static_assert(SORT_MAX % 32 == 0 && SORT_MAX >= 8192, "sorted walk must cover a 1024-word tile at 25 % density");
    uint32_t* s_wx = reinterpret_cast<uint32_t*>(s_stage + SORT_MAX);
    uint32_t* s_wm = s_wx + TILE_WORDS;
    __shared__ int s_bkt[33];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) s_tile = static_cast<int>(atomicAdd(status, 1ull));
    if (threadIdx.x < 33) s_bkt[threadIdx.x] = 0;
    __syncthreads();
    const int tile = s_tile;
    // all word indices fit 32 bits: rows * nk <= INT32_MAX is checked by the caller
    const uint32_t n_words = static_cast<uint32_t>(rows * words);
    const uint32_t tile0 = static_cast<uint32_t>(tile) * TILE_WORDS;
    const int rem = nk - (words - 1) * 32;                      // valid bits of a row's last word
    const uint32_t last_mask = rem >= 32 ? 0xffffffffu : ((1u << rem) - 1u);

    // 1. load WPT consecutive words per thread, mask the pad bits, count
    const uint32_t w0 = tile0 + threadIdx.x * WPT;              // this thread's first word
    uint32_t v[WPT];
    uint32_t fu[kGeo ? WPT : 1], fl[kGeo ? WPT : 1];            // kGeo: source bits of the two mask rows
    const uint32_t row0 = w0 / static_cast<uint32_t>(words);    // one division per thread and tile
    const int win0 = static_cast<int>(w0 - row0 * static_cast<uint32_t>(words));
    int cnt = 0;
    {
        int wr = win0;
        uint32_t r = row0;
#pragma unroll
        for (int i = 0; i < WPT; ++i) {
            uint32_t x = 0u;
            if constexpr (kGeo) {
                fu[i] = fl[i] = 0u;
                if (w0 + i < n_words) x = geo_word(geo, r, wr, fu[i], fl[i]);
            } else {
                if (w0 + i < n_words) x = __ldg(bitmask + w0 + i);
            }
            if (wr == words - 1) x &= last_mask;
            v[i] = x;
            cnt += __popc(x);
            if (++wr == words) { wr = 0; ++r; }
        }
    }
    // (histogram of the words' popcounts for the balanced walk below; complete at the next barrier)
    int rank[WPT];
#pragma unroll
    for (int i = 0; i < WPT; ++i) {
        const int pc = __popc(v[i]);
        rank[i] = (kSort && pc) ? atomicAdd(&s_bkt[32 - pc], 1) : 0;
    }
    // 2a/2b. one exclusive scan of the thread counts inside the block
    int inc = cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int u = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += u;
    }
    if (lane == 31) s_warp[warp] = inc;
    __syncthreads();
    int off = inc - cnt, tile_total = 0;     // set bits of the tile in front of this thread's words
#pragma unroll
    for (int w = 0; w < DEC_WARPS; ++w) {
        const int u = s_warp[w];
        if (w < warp) off += u;
        tile_total += u;
    }
    // a tile whose entries all fit the staging buffer is expanded in one go (the usual case)
    const bool fast = col_idx != nullptr && tile_total <= STAGE;
    // 2c. decoupled look-back, 256 predecessor tiles per step (thread i looks at tile look - i): with
    // a thousand tiles in flight the nearest tile that already knows its prefix is that far back
    {
        unsigned long long* mine = status + 1 + tile;
        if (threadIdx.x == 0)
            st_status(mine, (tile == 0 ? ST_INC : ST_AGG) | static_cast<uint32_t>(tile_total));
        // While the predecessors publish, expand: the staging offsets do not need the global base.
        // Balanced walk.  A warp walks as long as its fullest lane, and popcounts differ a lot (the all-kept frame-0
        // blocks of every row's first word, L81; binomial spread elsewhere): with every thread walking its own
        // words the tile costs 2.3 x the warp iterations of a balanced walk.  The tile's non-empty words are
        // therefore counting-sorted by popcount in shared memory (33 buckets, descending) and thread t walks the
        // sorted words t, t + 256, ...: the 32 lanes of a warp get words of (nearly) the same popcount.  A word
        // carries its staging offset and its position in the row along, so where it is walked does not matter.
        if (fast && kSort && tile_total <= SORT_MAX) {
            static_assert(STAGE <= (1 << 14), "staging offset must fit 14 bits");
            // every warp scans the 32 buckets (popcount 32, 31, .., 1) for itself: no second barrier
            const int c = s_bkt[lane];
            int incl = c;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int u = __shfl_up_sync(0xffffffffu, incl, o);
                if (lane >= o) incl += u;
            }
            const int start = incl - c;
            const int n_nz = __shfl_sync(0xffffffffu, incl, 31);   // non-empty words of the tile
            {
                int e = off, wr = win0;
#pragma unroll
                for (int i = 0; i < WPT; ++i) {
                    const int pc = __popc(v[i]);
                    const int st = __shfl_sync(0xffffffffu, start, (32 - pc) & 31);
                    if (pc) {
                        const int pos = st + rank[i];
                        s_wx[pos] = v[i];
                        s_wm[pos] = static_cast<uint32_t>(e) | (static_cast<uint32_t>(wr) << 14);
                    }
                    e += pc;
                    if (++wr == words) wr = 0;
                }
            }
            __syncthreads();
#pragma unroll
            for (int i = 0; i < WPT; ++i) {
                const int pos = i * DEC_THREADS + static_cast<int>(threadIdx.x);
                if (pos < n_nz) {
                    const uint32_t x = s_wx[pos], meta = s_wm[pos];
                    const int kb0 = static_cast<int>(meta >> 14) * 32;
                    walk_word(x, static_cast<int>(meta & 0x3fffu), s_stage, [&](int b) { return stage_entry<StageT, kGeo>(kb0 + b); });
                }
            }
        } else if (fast) {
            int e = off, wr = win0;
#pragma unroll
            for (int i = 0; i < WPT; ++i) {
                const int kb0 = wr * 32;
                if constexpr (kGeo) {
                    const uint32_t gu = fu[i], gl = fl[i];
                    walk_word(v[i], e, s_stage, [&](int b) { return stage_entry<StageT, kGeo>(geo_entry(kb0 + b, b, gu, gl)); });
                } else {
                    walk_word(v[i], e, s_stage, [&](int b) { return stage_entry<StageT, kGeo>(kb0 + b); });
                }
                e += __popc(v[i]);
                if (++wr == words) wr = 0;
            }
        }
        int base = 0;
        for (int look = tile - 1; tile > 0;) {
            const int t = look - static_cast<int>(threadIdx.x);
            unsigned long long sv = ST_INC;         // in front of tile 0: prefix 0
            if (t >= 0) {
                do { sv = ld_status(status + 1 + t); } while ((sv >> 62) == 0);
            }
            const unsigned inc_mask = __ballot_sync(0xffffffffu, (sv >> 62) == 2);
            const int first_inc = __ffs(inc_mask) - 1;              // nearest one in this warp's window
            const int val = (inc_mask == 0 || lane <= first_inc) ? static_cast<int>(sv & 0xffffffffu) : 0;
            const int wsum = __reduce_add_sync(0xffffffffu, val);
            __syncthreads();                        // s_look is free (previous step / s_warp users done)
            if (lane == 0) s_look[warp] = make_int2(wsum, inc_mask != 0);
            __syncthreads();
            bool done = false;
#pragma unroll
            for (int w = 0; w < DEC_WARPS; ++w) {   // warp 0 holds the nearest predecessors
                const int2 u = s_look[w];
                if (!done) base += u.x;
                done = done || (u.y != 0);
            }
            if (done) break;
            look -= DEC_THREADS;
        }
        if (tile > 0 && threadIdx.x == 0) st_status(mine, ST_INC | static_cast<uint32_t>(base + tile_total));
        if (threadIdx.x == 0) s_base = base;
    }
    __syncthreads();
    const int64_t base = s_base;
    // 3a. row_ptr of the rows that begin in this tile; the thread holding the last word writes the total
    {
        int o = off, wr = win0;
        uint32_t r = row0;
#pragma unroll
        for (int i = 0; i < WPT; ++i) {
            if (wr == 0 && w0 + i < n_words) row_ptr[r] = static_cast<int32_t>(base + o);
            if (w0 + i == n_words - 1) row_ptr[rows] = static_cast<int32_t>(base + tile_total);
            o += __popc(v[i]);
            if (++wr == words) { wr = 0; ++r; }
        }
    }
    if (col_idx == nullptr) return;
    if (fast) {     // staged before the look-back; the __syncthreads after it ordered the writes
        // entries beyond col_cap are never written: clamp once, then 32-bit indices only
        const int n_out = static_cast<int>(min(static_cast<int64_t>(tile_total), max(col_cap - base, static_cast<int64_t>(0))));
        IdxT* dst = col_idx + base;
#pragma unroll 4
        for (int t = threadIdx.x; t < n_out; t += DEC_THREADS) dst[t] = unstage_entry<IdxT, StageT, kGeo>(s_stage[slot(t)]);
        return;
    }
    // 3b. a fuller tile (WPT > 1 only): WPT rounds of one word per thread, so that every thread walks
    // in every round.  Round r takes words r*256 .. r*256+255 of the tile - at most 8192 entries, one
    // contiguous run - and finds each word's offset in a table the owning threads wrote; the table
    // sits behind the largest round in the staging buffer.
    if constexpr (WPT > 1) {
        constexpr int ROUND_MAX = DEC_THREADS * 32;
        static_assert(ROUND_MAX * sizeof(StageT) + TILE_WORDS * 4 <= sizeof(s_raw), "staging buffer too small for a round plus the offset table");
        int* s_woff = reinterpret_cast<int*>(s_raw + ROUND_MAX * sizeof(StageT));
        {
            int o = off;
#pragma unroll
            for (int i = 0; i < WPT; ++i) {
                s_woff[threadIdx.x * WPT + i] = o;
                o += __popc(v[i]);
            }
        }
        __syncthreads();
#pragma unroll 1
        for (int r = 0; r < WPT; ++r) {
            const int j = r * DEC_THREADS + threadIdx.x;
            const int lo = s_woff[r * DEC_THREADS];
            const int hi = r + 1 < WPT ? s_woff[(r + 1) * DEC_THREADS] : tile_total;
            const uint32_t g = tile0 + j;
            const uint32_t gr = g / static_cast<uint32_t>(words);
            const int wr = static_cast<int>(g - gr * static_cast<uint32_t>(words));
            uint32_t x = 0u, gu = 0u, gl = 0u;
            if (g < n_words) x = kGeo ? geo_word(geo, gr, wr, gu, gl) : __ldg(bitmask + g);
            if (wr == words - 1) x &= last_mask;
            const int e = s_woff[j] - lo;
            const int kb0 = wr * 32;
            if constexpr (kGeo) walk_word(x, e, s_stage, [&](int b) { return stage_entry<StageT, kGeo>(geo_entry(kb0 + b, b, gu, gl)); });
            else walk_word(x, e, s_stage, [&](int b) { return stage_entry<StageT, kGeo>(kb0 + b); });
            __syncthreads();
            const int n_out = static_cast<int>(min(static_cast<int64_t>(hi - lo), max(col_cap - base - lo, static_cast<int64_t>(0))));
            IdxT* dst = col_idx + base + lo;
#pragma unroll 4
            for (int t = threadIdx.x; t < n_out; t += DEC_THREADS) dst[t] = unstage_entry<IdxT, StageT, kGeo>(s_stage[slot(t)]);
            __syncthreads();
        }
    }
}

// Visit refresh (PAPER.md:L93 (1)): one thread per (group, word of a layer).
__global__ void __launch_bounds__(256)
visit_refresh_kernel(uint32_t* __restrict__ bitmask, int n_groups, int64_t words_per_layer,
                     int words, int nk, int group) {
    const int64_t total = static_cast<int64_t>(n_groups) * words_per_layer;
    for (int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x; i < total;
         i += static_cast<int64_t>(gridDim.x) * blockDim.x) {
        const int64_t g = i / words_per_layer, x = i - g * words_per_layer;
        uint32_t* base = bitmask + (g * group) * words_per_layer + x;
        uint32_t seen = 0u;
        for (int l = 0; l < group - 1; ++l) seen |= base[l * words_per_layer];
        const int w = static_cast<int>(x % words);
        const int rem = nk - w * 32;
        const uint32_t valid = rem >= 32 ? 0xffffffffu : (rem <= 0 ? 0u : ((1u << rem) - 1u));
        base[(group - 1) * words_per_layer] |= (~seen) & valid;
    }
}

// one word per thread below this many words (a few layers), four above
constexpr int64_t SMALL_WORDS = 1 << 20;
inline int wpt_for(int64_t n_words) { return n_words < SMALL_WORDS ? 1 : 4; }
inline int64_t n_tiles_for(int64_t rows, int words) {
    const int64_t n = rows * words, tw = static_cast<int64_t>(DEC_THREADS) * wpt_for(n);
    return (n + tw - 1) / tw;
}

}  // namespace

size_t decode_workspace_bytes(int64_t rows, int words) {
    // ticket counter + one status word per tile, + 8 so that the array can be 8-byte aligned
    return static_cast<size_t>(n_tiles_for(rows, words) + 1) * sizeof(unsigned long long) + 8;
}

template <int V> struct IntTag { static constexpr int value = V; };
template <bool V> struct BoolTag { static constexpr bool value = V; };
template <typename T> struct TypeTag { using type = T; };

template <typename IdxT>
static cudaError_t launch_decode(const uint32_t* bitmask, const GeoSrc* geo, int64_t rows, int nk, int words,
                                 int32_t* row_ptr, IdxT* col_idx, int64_t col_cap, void* workspace,
                                 cudaStream_t stream) {
    const int64_t nt = n_tiles_for(rows, words);
    auto* status = reinterpret_cast<unsigned long long*>((reinterpret_cast<uintptr_t>(workspace) + 7) & ~uintptr_t(7));
    cudaError_t e = cudaMemsetAsync(status, 0, static_cast<size_t>(nt + 1) * sizeof(unsigned long long), stream);
    if (e != cudaSuccess) return e;
    const unsigned grid = static_cast<unsigned>(nt);
    const bool one = wpt_for(rows * words) == 1;
    const GeoSrc g = geo ? *geo : GeoSrc{nullptr, 0, 0, 0, 0};
    // entries that fit 16 bits are staged in 16-bit slots: always for 16-bit output; for 32-bit output when they carry
    // no flags (plain geometry) and nk <= 65536
    auto go = [&](auto wpt_tag, auto geo_tag, auto stage_tag) {
        constexpr int W = decltype(wpt_tag)::value;
        constexpr bool G = decltype(geo_tag)::value;
        using StageT = typename decltype(stage_tag)::type;
        decode_tiles_kernel<W, G, IdxT, StageT><<<grid, DEC_THREADS, 0, stream>>>(geo ? nullptr : bitmask, rows, nk, words, row_ptr,
                                                                                col_idx, col_cap, status, g);
    };
    const bool stage16 = sizeof(IdxT) == 2 || (!geo && nk <= 65536);
    if (geo) {
        if constexpr (sizeof(IdxT) == 2) {
            if (one) go(IntTag<1>{}, BoolTag<true>{}, TypeTag<uint16_t>{});
            else go(IntTag<4>{}, BoolTag<true>{}, TypeTag<uint16_t>{});
        } else {
            if (one) go(IntTag<1>{}, BoolTag<true>{}, TypeTag<int32_t>{});
            else go(IntTag<4>{}, BoolTag<true>{}, TypeTag<int32_t>{});
        }
    } else if (stage16) {
        if (one) go(IntTag<1>{}, BoolTag<false>{}, TypeTag<uint16_t>{});
        else go(IntTag<4>{}, BoolTag<false>{}, TypeTag<uint16_t>{});
    } else {
        if constexpr (sizeof(IdxT) == 4) {
            if (one) go(IntTag<1>{}, BoolTag<false>{}, TypeTag<int32_t>{});
            else go(IntTag<4>{}, BoolTag<false>{}, TypeTag<int32_t>{});
        }
    }
    count_launch(1);
    return cudaGetLastError();
}

cudaError_t launch_mask_decode(const uint32_t* bitmask, int64_t rows, int nk, int words,
                               int32_t* row_ptr, void* col_idx, bool idx16, int64_t col_cap, void* workspace,
                               cudaStream_t stream) {
    if (idx16)
        return launch_decode<uint16_t>(bitmask, nullptr, rows, nk, words, row_ptr, static_cast<uint16_t*>(col_idx), col_cap, workspace, stream);
    return launch_decode<int32_t>(bitmask, nullptr, rows, nk, words, row_ptr, static_cast<int32_t*>(col_idx), col_cap, workspace, stream);
}

// ---- decode without any allocation (chorus_mask_to_index_static) --------------------------------------------------
// For callers that cannot provide or allocate a workspace (CUDA graph capture, serving loops and harnesses that
// forbid cudaMalloc): the per-tile status words live in this file-scope device array, 128 KB that every GPU which
// loads the library holds until exit.  All calls share it, so two such calls that overlap on the GPU race; it keeps
// the previous call's contents, and launch_decode clears the words it is going to use (a memset node on the call's
// stream, no allocation) as it does with a caller's workspace.
static __device__ __align__(256) unsigned long long g_decode_scratch[STATIC_DECODE_MAX_TILES + 1];

int64_t decode_static_tiles(int64_t rows, int words) { return n_tiles_for(rows, words); }

// In host code `g_decode_scratch` is a host-side stand-in, not a device address: the address is asked for once per
// device, with that device current, and kept.
static cudaError_t decode_scratch_address(unsigned long long** out) {
    constexpr int MAX_DEVICES = 64;
    static std::mutex mu;
    static unsigned long long* addr[MAX_DEVICES] = {};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(mu);
    if (!addr[dev]) {
        void* ptr = nullptr;
        e = cudaGetSymbolAddress(&ptr, g_decode_scratch);
        if (e != cudaSuccess) return e;
        if (!ptr || (reinterpret_cast<uintptr_t>(ptr) & 255u)) return cudaErrorInvalidSymbol;
        addr[dev] = static_cast<unsigned long long*>(ptr);
    }
    *out = addr[dev];
    return cudaSuccess;
}

cudaError_t launch_mask_decode_static(const uint32_t* bitmask, int64_t rows, int nk, int words, int32_t* row_ptr,
                                      void* col_idx, bool idx16, int64_t col_cap, cudaStream_t stream) {
    if (n_tiles_for(rows, words) > STATIC_DECODE_MAX_TILES) return cudaErrorInvalidValue;   // (checked by the caller)
    unsigned long long* scratch = nullptr;
    cudaError_t e = decode_scratch_address(&scratch);
    if (e != cudaSuccess) return e;
    if (idx16)
        return launch_decode<uint16_t>(bitmask, nullptr, rows, nk, words, row_ptr, static_cast<uint16_t*>(col_idx), col_cap, scratch, stream);
    return launch_decode<int32_t>(bitmask, nullptr, rows, nk, words, row_ptr, static_cast<int32_t*>(col_idx), col_cap, scratch, stream);
}

cudaError_t launch_visit_refresh(uint32_t* bitmask, int L, int64_t words_per_layer, int words,
                                 int nk, int group, cudaStream_t stream) {
    const int n_groups = L / group;
    if (n_groups == 0) return cudaSuccess;
    const int64_t total = static_cast<int64_t>(n_groups) * words_per_layer;
    const int blocks = static_cast<int>(std::min<int64_t>((total + 255) / 256, 148 * 16));
    visit_refresh_kernel<<<blocks, 256, 0, stream>>>(bitmask, n_groups, words_per_layer, words, nk,
                                                     group);
    count_launch(1);
    return cudaGetLastError();
}

size_t decode_64x128_workspace_bytes(int64_t heads, int N) {
    const int nq128 = (N + 127) / 128, words64 = ((N + 63) / 64 + 31) / 32;
    return decode_workspace_bytes(heads * nq128, words64);
}

// One launch: the decode kernel reads the 64 x 128 mask rows directly (GeoSrc) and writes the flagged entries.
cudaError_t launch_mask_decode_64x128(const uint32_t* bm64, int64_t heads, int N, int32_t* row_ptr,
                                      void* col_idx, bool idx16, int64_t col_cap, void* workspace, cudaStream_t stream) {
    const int nq64 = (N + 63) / 64, nq128 = (N + 127) / 128, nk128 = nq128, nk64 = nq64;
    const GeoSrc geo{bm64, nq64, nq128, nk128, (nk128 + 31) / 32};
    if (idx16)
        return launch_decode<uint16_t>(nullptr, &geo, heads * nq128, nk64, (nk64 + 31) / 32, row_ptr,
                                       static_cast<uint16_t*>(col_idx), col_cap, workspace, stream);
    return launch_decode<int32_t>(nullptr, &geo, heads * nq128, nk64, (nk64 + 31) / 32, row_ptr,
                                  static_cast<int32_t*>(col_idx), col_cap, workspace, stream);
}

}  // namespace chorus
