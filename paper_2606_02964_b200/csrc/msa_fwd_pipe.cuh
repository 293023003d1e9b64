// msa_fwd_pipe: the warp-specialised, pipelined MSA forward kernel for sm_100a.
//
// One persistent CTA per SM (512 threads), roles by warp:
//   warps 0-3   softmax warpgroup of chain 0   (one thread per packed (head, token) row)
//   warps 4-7   softmax warpgroup of chain 1
//   warps 8-11  epilogue warpgroup (O / l -> bf16, LSE, split-KV partials; in-CTA merge)
//   warp  12    loader of Q and K tiles: virtual blocks -> TMA boxes (paged and contiguous alike)
//   warp  13    MMA issuer: tcgen05.mma for S = Q K^T and O += P V, accumulators in TMEM
//   warp  14    loader of V tiles (same code path as warp 12)
//   warp  15    write-back warp in a write-back launch (msa_forward_writeback), else idle
//
// KV8 variant (fp8 E4M3 paged pool): cached blocks arrive as bytes in a staging ring (warp 15 issues
// their TMA boxes), warps 8-11 turn them into the bf16 rows of the tile's ring slot (exact: code * 2^k) before they
// do the unit's epilogue, and warps 12 / 14 load only the arena blocks of a tile directly; a ring slot is "full" once
// the loader and the four converter warps have arrived.  The MMA and softmax roles are the same code in both variants.
//
// Two independent "chains" keep the tensor core busy while the other chain's softmax runs:
//   kModePair   chain c owns q tile c of the unit; both chains consume every KV tile
//   kModeSplit  one q tile; chain c owns KV tiles c, c+2, ... with its own (ref, l, O);
//               the epilogue merges the two partial softmaxes (short / decode-like queries)
// TMEM (512 columns): S0 [0,128) S1 [128,256) O0 [256,384) O1 [384,512); P (bf16) aliases
// the first 64 columns of its S and is handed to the MMA warp in three parts (keys 0-63, 64-95,
// 96-127), so that O += P V trails the exponentials.
// Shared memory: Q 2 tiles, one ring of 5 tile slots in which K and V tiles alternate (entry
// 2i = K of the CTA's i-th KV tile, 2i+1 = its V).  The softmax arithmetic, its integer row
// reference and the overflow guard of the fast path are described in msa_softmax.cuh.
//
// Invalid KV slots (block tails, blocks past a context's end or past the causal horizon) never
// reach O: their scores are replaced by -inf (P = 0), their K/V rows are never written by TMA --
// partly filled blocks load through 8/4/2/1-row boxes -- and the V loader zeroes exactly those
// rows of its ring slot before it arms the tile, so P = 0 never meets stale data (another
// request's Inf / NaN would otherwise turn 0 * x into NaN).
#pragma once
#include <math.h>

#include "msa_kernels.h"
#include "msa_ptx.cuh"
#include "msa_softmax.cuh"
#include "msa_kv8.cuh"
#include "msa_prof.cuh"      // PROF_* hooks: empty unless built with -DMSA_PROF (never the shipped library)

namespace msa {

template <int D, bool KV8 = false, int QT = 2>
struct PipeCfg {
    static constexpr int kHalves = D / 64;
    static constexpr int kHalfBytes = kTileM * 128;                  // 128 rows x 128 B
    static constexpr int kTileBytes = kHalves * kHalfBytes;
    static constexpr int kStages = KV8 ? 4 : 5;
    static constexpr int kQBytes = QT * kTileBytes;                  // QT = 1: a launch without pair-mode units (short queries only)
    static constexpr int kRingBytes = kStages * kTileBytes;
    // KV8: staging ring for the fp8 blocks of a tile (128 rows x D bytes, row-major, no swizzle).  It holds the fp8
    // bytes that are in flight from HBM; the bf16 ring behind it only decouples converters and tensor core.  A
    // short-query launch needs one Q tile and spends the other's room on two more staging slots (an SM's share of the
    // HBM stream in flight); a launch with prefill units reuses every K/V tile 256 rows long and needs little in flight.
    static constexpr int kStgStages = KV8 ? (QT == 1 ? 4 : 2) : 0;
    static constexpr int kStgDiv = kStgStages ? kStgStages : 1;      // (keeps the dead staging code of the bf16 variant well formed)
    static constexpr int kStgTileBytes = kTileN * D;
    static constexpr int kStgBytes = kStgStages * kStgTileBytes;
    static constexpr int kStatsBytes = 2 * kTileM * 2 * 4;           // [chain][row]{l, m}
    static constexpr int kBarBytes = 512;
    static constexpr int kSmemBytes = kQBytes + kRingBytes + kStgBytes + kStatsBytes + kBarBytes;
    static constexpr uint32_t kColS = 0, kColO = 256, kChainCols = 128;
    static constexpr float kRescaleThreshold = 8.0f;                 // log2 units (lazy rescale)
};

enum PipeBar : int {
    kBarQFull = 0, kBarQEmpty = 1,
    kBarKvFull = 2,      // [5]
    kBarKvEmpty = 7,     // [5]
    kBarSFull = 12,      // [2]
    kBarPLo = 14,        // [2] P of keys 0-63 in TMEM
    kBarOFull = 16,      // [2]
    kBarOFree = 18,      // [2]
    // 20, 21: free (the stats hand-off is a named barrier: the epilogue warps wait for a whole unit)
    kBarStFree = 22,     // [2]
    kBarPQ2 = 24,        // [2] P of keys 64-95 in TMEM
    kBarPQ3 = 26,        // [2] P of keys 96-127 in TMEM
    kBarStgFull = 28,    // [4] KV8: fp8 blocks of a K (or V) tile have landed in a staging slot
    kBarStgEmpty = 32,   // [4] KV8: the four converter warps are done with a staging slot
    kBarQReady = 36,     // f16 variant: the converter warps have turned the unit's Q tile into f16
    kBarKvDirect = 37,   // [5] f16 variant: the arena (bf16) blocks of a ring slot have landed and wait for their conversion
    kBarCount = 42
};
constexpr int kConvWarps = 4;          // KV8: warps 8-11 convert (and, per unit, do the epilogue)

constexpr bool kWritebackRing = true;  // the ring's "empty" barriers take a second arrival (the loader, or the write-back warp)
constexpr uint32_t kNamedStFull = 1;   // named barriers 1, 2: (l, ref) of chain 0 / 1 are in shared memory (128 + 128 threads)

struct RingPos {
    uint32_t slot, phase;
    __device__ __forceinline__ void advance2(int stages)   // K and V entries alternate in the ring
    {
        slot += 2;
        if (slot >= static_cast<uint32_t>(stages)) {
            slot -= stages;
            phase ^= 1;
        }
    }
};

// KV8: the ring holds the tiles of a unit in the order the MMA warp takes them, so that an entry's slot is free again
// a fixed number of entries later whatever the mode:
//   pair mode   K0 V0 K1 V1 ...                          (K(j+1) is taken while V(j) is being multiplied)
//   split mode  K0 K1 V0 K2 V1 ... K(n-1) V(n-2) V(n-1)  (QK of tile j+2 follows PV of tile j)
// Index of K(i) / V(j) in that order, and its inverse.
__device__ __forceinline__ int kv8_entry_of_k(int i, bool pair)
{
    return pair ? 2 * i : (i < 2 ? i : 2 * i - 1);
}
__device__ __forceinline__ int kv8_entry_of_v(int j, int n, bool pair)
{
    return pair ? 2 * j + 1 : (j == n - 1 ? 2 * n - 1 : 2 * j + 2);
}
__device__ __forceinline__ void kv8_entry(int e, int n, bool pair, bool &is_v, int &tile)
{
    if (pair) {
        is_v = (e & 1) != 0;
        tile = e >> 1;
    } else if (e == 0) {
        is_v = false;
        tile = 0;
    } else if (e == 2 * n - 1) {
        is_v = true;
        tile = n - 1;
    } else if (e & 1) {
        is_v = false;
        tile = (e + 1) >> 1;
    } else {
        is_v = true;
        tile = (e - 2) >> 1;
    }
}

struct ResolvedVb {
    int32_t row;      // first row in the pool / arena row space
    int32_t nvp;      // valid slots (0: nothing to load) | paged << 8
};

// The fp8 blocks of one K (or V) tile: staging slot (row-major, D bytes per row, block b at b*16*D) -> the bf16 tile in
// its ring slot (128-byte swizzle, one 16 KB half per 64 elements, as TMA would have written it).  A warp iteration
// covers 512 staged bytes (a lane: 16 codes = two 16-byte bf16 chunks); the calling warp takes the iterations whose bit
// is set in it_mask (even_w >= 0: the mask is the even split's, warp even_w of four).  Only rows < nvalid of a block are written (the V loader has zeroed the others, K's are masked).
// The two stores of the lanes j and j + 4 of a row go to the same bank group (different 64-element halves): a two-way
// conflict on the store pipe, which has room; ordering the stores per lane to avoid it costs ten selects per iteration
// on the ALU pipe, which is what bounds the conversion (measured).
template <int D, bool F16 = false>
__device__ __forceinline__ void kv8_convert_tile(uint32_t stg, uint32_t dst, uint32_t m_paged, int nvp, uint32_t mul,
                                                 uint32_t it_mask, int even_w, int lane)
{
    constexpr int kLanesPerRow = D / 16, kRowsPerIt = 32 / kLanesPerRow, kItPerBlock = kBlock / kRowsPerIt;
    constexpr int kHalfBytes = kTileM * 128;
    const int chunk = lane % kLanesPerRow, rsub = lane / kLanesPerRow;
    const uint32_t c0 = static_cast<uint32_t>(2 * (chunk & 3));
    const uint32_t src0 = stg + static_cast<uint32_t>(rsub * D + chunk * 16);
    const uint32_t dst0 = dst + static_cast<uint32_t>((chunk >> 2) * kHalfBytes + rsub * 128);
    constexpr int kIters = kVbPerTile * kItPerBlock;
    const uint32_t mul2 = (mul & 0xffffu) * 0x10001u;      // f16 bits of 2^k in both halves
    auto convert_store = [&](int it, uint32_t w0, uint32_t w1, uint32_t w2, uint32_t w3) {
        const int row0 = (it / kItPerBlock) * kBlock + (it % kItPerBlock) * kRowsPerIt;      // tile row of the iteration's first row
        const uint32_t base = dst0 + static_cast<uint32_t>(row0 * 128);
        const uint32_t x = static_cast<uint32_t>((row0 + rsub) & 7);
        // code * 2^k, exactly: as f16 (F16: one cvt and one packed multiply per pair) or as bf16
        auto cv = [mul, mul2](uint32_t two) { return F16 ? e4m3x2_to_f16x2(two, mul2) : e4m3x2_to_bf16x2(two, mul); };
        const uint32_t o0 = cv(w0), o1 = cv(w0 >> 16), o2 = cv(w1), o3 = cv(w1 >> 16);
        const uint32_t o4 = cv(w2), o5 = cv(w2 >> 16), o6 = cv(w3), o7 = cv(w3 >> 16);
        asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(base + ((c0 ^ x) << 4)), "r"(o0), "r"(o1), "r"(o2), "r"(o3) : "memory");
        asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(base + (((c0 + 1) ^ x) << 4)), "r"(o4), "r"(o5), "r"(o6), "r"(o7) : "memory");
    };
    auto load = [&](int it, uint32_t &w0, uint32_t &w1, uint32_t &w2, uint32_t &w3) {
        const int row0 = (it / kItPerBlock) * kBlock + (it % kItPerBlock) * kRowsPerIt;
        asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];"
                     : "=r"(w0), "=r"(w1), "=r"(w2), "=r"(w3)
                     : "r"(src0 + static_cast<uint32_t>(row0 * D)));
    };
    const bool all_full = m_paged == 0xffu && __all_sync(0xffffffffu, lane >= kVbPerTile || (nvp & 0xff) == kBlock);
    if (all_full && even_w >= 0) {
        // The common tile (eight full cached blocks), iterations dealt out evenly: warp w takes w, w + 4, ...  Four
        // iterations further on is 2048 staged bytes and a whole number of 8-row swizzle groups further on, so a lane's load
        // and store addresses are its first ones plus compile-time constants: nothing but the loads, the conversions and the
        // stores is left in the unrolled loop (a warp instruction of the integer pipe issues every other cycle, and the
        // address arithmetic of the general loop below costs more of them than the conversion itself).
        constexpr int kPerWarp = kIters / kConvWarps;
        constexpr uint32_t kSrcStep = 4u * kRowsPerIt * D, kDstStep = 4u * kRowsPerIt * 128u;
        const int row_w = (even_w / kItPerBlock) * kBlock + (even_w % kItPerBlock) * kRowsPerIt + rsub;
        const uint32_t x = static_cast<uint32_t>(row_w & 7);
        const uint32_t src_l = stg + static_cast<uint32_t>(row_w * D + chunk * 16);
        const uint32_t dst_l = dst + static_cast<uint32_t>((chunk >> 2) * kHalfBytes + row_w * 128);
        // The lanes j and j + 4 of a row write the same bank group (different 64-element halves): the upper four store their two
        // chunks in the other order, so that the eight lanes of a quarter-warp hit eight different bank groups (the conversion is
        // bound by the shared-memory pipe: a two-way conflict on every store costs a third of its time)
        const bool sw = kLanesPerRow == 8 && (chunk & 4) != 0;
        const uint32_t da = dst_l + ((c0 ^ x) << 4), db = dst_l + (((c0 + 1) ^ x) << 4);
        const uint32_t d0 = sw ? db : da, d1 = sw ? da : db;
        auto cv = [mul, mul2](uint32_t two) { return F16 ? e4m3x2_to_f16x2(two, mul2) : e4m3x2_to_bf16x2(two, mul); };
#pragma unroll
        for (int k0 = 0; k0 < kPerWarp; k0 += 4) {
            uint32_t w[4][4];
#pragma unroll
            for (int k = 0; k < 4; ++k)
                if (k0 + k < kPerWarp)
                    asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];"
                                 : "=r"(w[k][0]), "=r"(w[k][1]), "=r"(w[k][2]), "=r"(w[k][3])
                                 : "r"(src_l + (k0 + k) * kSrcStep));
#pragma unroll
            for (int k = 0; k < 4; ++k)
                if (k0 + k < kPerWarp) {
                    // (the codes are swapped, not the converted values: two selects per store)
                    const uint32_t a0 = sw ? w[k][2] : w[k][0], a1 = sw ? w[k][3] : w[k][1];
                    const uint32_t b0 = sw ? w[k][0] : w[k][2], b1 = sw ? w[k][1] : w[k][3];
                    asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(d0 + (k0 + k) * kDstStep), "r"(cv(a0)),
                                 "r"(cv(a0 >> 16)), "r"(cv(a1)), "r"(cv(a1 >> 16)) : "memory");
                    asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(d1 + (k0 + k) * kDstStep), "r"(cv(b0)),
                                 "r"(cv(b0 >> 16)), "r"(cv(b1)), "r"(cv(b1 >> 16)) : "memory");
                }
        }
        return;
    }
#pragma unroll 1
    while (it_mask != 0) {
        const int it = __ffs(it_mask) - 1;
        it_mask &= it_mask - 1;
        const int b = it / kItPerBlock;
        const int nv = __shfl_sync(0xffffffffu, nvp, b) & 0xff;
        if (((m_paged >> b) & 1u) && (it % kItPerBlock) * kRowsPerIt + rsub < nv) {
            uint32_t w0, w1, w2, w3;
            load(it, w0, w1, w2, w3);
            convert_store(it, w0, w1, w2, w3);
        }
    }
}

// KV8 converters (warps 8-11): every ring entry of the unit in ring order; for an entry whose tile holds cached blocks,
// the calling warp converts the iterations of its mask (kv8_convert_tile) of the staged codes into the tile's ring slot
// and arrives on the staging slot's "empty" barrier; every warp arrives on the ring slot's "full"
// barrier for every entry.  An entry is waited for even when there is nothing to convert: a waiter that skips a use
// of a slot cannot tell the phases of its barrier apart.
// f16 variant: 16-byte chunks [first, n) in steps of stride * 32 of a shared-memory region, bf16 -> f16 in place (exact for
// magnitudes in [2^-14, 65504]; beyond +-65504 it saturates, below 2^-14 the value is rounded to a multiple of 2^-24).
__device__ __forceinline__ void bf16_to_f16_inplace(uint32_t base, int n_chunks, int first, int stride, int lane)
{
    for (int i = first * 32 + lane; i < n_chunks; i += stride * 32) {
        uint32_t w[4];
        asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(w[0]), "=r"(w[1]), "=r"(w[2]), "=r"(w[3]) : "r"(base + i * 16u));
#pragma unroll
        for (int k = 0; k < 4; ++k)
            w[k] = pack_f16x2_sat(__uint_as_float(w[k] << 16), __uint_as_float(w[k] & 0xffff0000u));
        asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(base + i * 16u), "r"(w[0]), "r"(w[1]), "r"(w[2]), "r"(w[3]) : "memory");
    }
}

// F16 (the short-query variant, see the kernel): the ring holds f16 tiles.  The codes become code * 2^k in f16 (exact for
// every legal scale), the arena blocks of a tile -- loaded as bf16 by the ring loaders, complete on the slot's "direct"
// barrier -- are rewritten in place as f16, and at the start of the unit the Q tile is rewritten as f16 (cw_first / cw_stride:
// this warp's share of that work; cw_first < 0: none).
template <class C, int D, bool F16>
__device__ __forceinline__ void kv8_convert_unit(const FwdParams &P, const WorkUnit &wu, uint32_t bar0, uint32_t sQ, uint32_t sStg,
                                                 uint32_t sRing, int lane, uint32_t it_mask, int even_w, int cw_first, int cw_stride,
                                                 uint32_t &cv_ent, uint32_t &cv_stg, uint32_t &cv_phq, uint32_t &dir_par, bool trace = false)
{
#if defined(MSA_PROF) && MSA_PROF == 2
#define CV_TRACE(step, ev) do { if (trace && (step) < 64) g_trace[3][step][ev] = clock64(); } while (0)
#else
#define CV_TRACE(step, ev)
    (void)trace;
#endif
    auto bar = [bar0](int i) { return bar0 + static_cast<uint32_t>(i) * 8u; };
    const int n = wu.tile_end - wu.tile_begin;
    const bool pair = wu.mode == kModePair;
    const uint32_t mul_k = __ldg(P.kv8_mul + wu.kvh), mul_v = __ldg(P.kv8_mul + P.Hkv + wu.kvh);
    PROF_DECL();
    if constexpr (F16) {
        if (n <= 0) return;
        // Q: bf16 -> f16 in place (the rows that hold tokens; all of them with head-major packing), then "Q ready"
        PROF_T0();
        mbar_wait(bar(kBarQFull), cv_phq);
        cv_phq ^= 1;
        const int rows_q = P.token_major ? min(kTileM, (wu.n_tok * P.G + 31) & ~31) : kTileM;     // whole softmax warps
        if (cw_first >= 0) {
#pragma unroll 1
            for (int h = 0; h < C::kHalves; ++h) bf16_to_f16_inplace(sQ + h * C::kHalfBytes, rows_q * 8, cw_first, cw_stride, lane);
        }
        fence_proxy_async_smem();
        __syncwarp();
        if (lane == 0) mbar_arrive(bar(kBarQReady));
        PROF_ADD(30);
    }
    auto fetch_nvp = [&](int e) -> int {             // lane b < 8: nvalid | paged << 8 of virtual block b of entry e's tile
        int r = 0;
        if (e < 2 * n) {
            bool is_v;
            int t;
            kv8_entry(e, n, pair, is_v, t);
            const int tile = wu.tile_begin + t;
            if (lane < kVbPerTile && tile * kVbPerTile + lane < wu.vb_count) {
                const int4 v = __ldg(reinterpret_cast<const int4 *>(P.vblocks + wu.vb_begin + tile * kVbPerTile + lane));
                r = v.z | ((v.z > 0 && v.w != 0) ? 256 : 0);
            }
        }
        return r;
    };
    int cur = fetch_nvp(0);
#pragma unroll 1
    for (int e = 0; e < 2 * n; ++e) {
        const int nxt = fetch_nvp(e + 1);
        const uint32_t m_paged = __ballot_sync(0xffffffffu, (cur >> 8) != 0) & 0xffu;
        const uint32_t m_dir = __ballot_sync(0xffffffffu, (cur >> 8) == 0 && (cur & 0xff) != 0) & 0xffu;
        bool is_v;
        int t;
        kv8_entry(e, n, pair, is_v, t);
        const uint32_t slot = cv_ent % C::kStages;
        {
            PROF_T0();
            mbar_wait(bar(kBarKvEmpty + slot), ((cv_ent / C::kStages) & 1u) ^ 1u);
            PROF_ADD(21);
        }
        CV_TRACE(e, 0);
        if (m_paged != 0) {
            const uint32_t st = cv_stg % static_cast<uint32_t>(C::kStgDiv);
            {
                PROF_T0();
                mbar_wait(bar(kBarStgFull + st), (cv_stg / C::kStgDiv) & 1u);
                PROF_ADD(22);
            }
            CV_TRACE(e, 1);
            PROF_T0();
            kv8_convert_tile<D, F16>(sStg + st * C::kStgTileBytes, sRing + slot * C::kTileBytes, m_paged, cur, is_v ? mul_v : mul_k,
                                     it_mask, even_w, lane);
            PROF_ADD(27);
            PROF_INC(24, 1);
            fence_proxy_async_smem();
            __syncwarp();
            if (lane == 0) mbar_arrive(bar(kBarStgEmpty + st));
            ++cv_stg;
        }
        if constexpr (F16) {
            // the arena blocks (and the V loader's zero fill) of this entry, if it has any, are in the slot
            const uint32_t m_full = __ballot_sync(0xffffffffu, (cur & 0xff) == kBlock) & 0xffu;
            if (m_dir != 0 || (is_v && m_full != 0xffu)) {
                PROF_T0();
                mbar_wait(bar(kBarKvDirect + slot), (dir_par >> slot) & 1u);
                PROF_ADD(28);
                dir_par ^= 1u << slot;
            }
            PROF_T0();
            if (m_dir != 0 && cw_first >= 0) {
                const uint32_t tile = sRing + slot * C::kTileBytes;
                if (m_dir == 0xffu && m_full == 0xffu && cw_stride == kConvWarps) {
                    // a tile of eight full arena blocks (the inside of a recomputed run): the whole slot, flat -- the 64-element
                    // halves follow each other -- in 16-byte chunks, a warp's share interleaved with the others', four loads in
                    // flight, every address a constant away from the lane's first
                    constexpr int kChunks = C::kTileBytes / 16, kPerLane = kChunks / (kConvWarps * 32);
                    const uint32_t a0 = tile + static_cast<uint32_t>((cw_first * 32 + lane) * 16);
#pragma unroll
                    for (int k0 = 0; k0 < kPerLane; k0 += 4) {
                        uint32_t w[4][4];
#pragma unroll
                        for (int k = 0; k < 4; ++k)
                            asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(w[k][0]), "=r"(w[k][1]), "=r"(w[k][2]), "=r"(w[k][3])
                                         : "r"(a0 + (k0 + k) * (kConvWarps * 32 * 16)));
#pragma unroll
                        for (int k = 0; k < 4; ++k) {
#pragma unroll
                            for (int j = 0; j < 4; ++j)
                                w[k][j] = pack_f16x2_sat(__uint_as_float(w[k][j] << 16), __uint_as_float(w[k][j] & 0xffff0000u));
                            asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(a0 + (k0 + k) * (kConvWarps * 32 * 16)), "r"(w[k][0]),
                                         "r"(w[k][1]), "r"(w[k][2]), "r"(w[k][3]) : "memory");
                        }
                    }
                } else
#pragma unroll 1
                for (int b = 0; b < kVbPerTile; ++b) {
                    if (!((m_dir >> b) & 1u)) continue;
                    const int nv = __shfl_sync(0xffffffffu, cur, b) & 0xff;
                    if (nv == kBlock && cw_stride == kConvWarps) {
                        // a full block: 16 rows x 128 B per 64-element half; the four warps take equal, fixed shares
                        constexpr int kChunks = kBlock * 8 * C::kHalves;         // 16-byte chunks of the block
                        constexpr int kPerLane = kChunks / (kConvWarps * 32);     // 2 (D = 128) or 1 (D = 64)
                        uint32_t w[kPerLane][4], addr[kPerLane];
#pragma unroll
                        for (int k = 0; k < kPerLane; ++k) {
                            const int i = (cw_first * kPerLane + k) * 32 + lane;  // chunk of the block, halves one after the other
                            addr[k] = tile + static_cast<uint32_t>((i / (kBlock * 8)) * C::kHalfBytes + b * (kBlock * 128) + (i % (kBlock * 8)) * 16);
                            asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(w[k][0]), "=r"(w[k][1]), "=r"(w[k][2]), "=r"(w[k][3]) : "r"(addr[k]));
                        }
#pragma unroll
                        for (int k = 0; k < kPerLane; ++k) {
#pragma unroll
                            for (int j = 0; j < 4; ++j)
                                w[k][j] = pack_f16x2_sat(__uint_as_float(w[k][j] << 16), __uint_as_float(w[k][j] & 0xffff0000u));
                            asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr[k]), "r"(w[k][0]), "r"(w[k][1]), "r"(w[k][2]), "r"(w[k][3]) : "memory");
                        }
                    } else {
#pragma unroll 1
                        for (int h = 0; h < C::kHalves; ++h)
                            bf16_to_f16_inplace(tile + h * C::kHalfBytes + b * (kBlock * 128), nv * 8, cw_first, cw_stride, lane);
                    }
                }
                fence_proxy_async_smem();
            }
            PROF_ADD(29);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(bar(kBarKvFull + slot));
        CV_TRACE(e, 2);
        ++cv_ent;
        cur = nxt;
    }
#if defined(MSA_PROF) && MSA_PROF != 2
#ifndef MSA_PROF_CVWARP
#define MSA_PROF_CVWARP 8
#endif
    if ((threadIdx.x >> 5) == MSA_PROF_CVWARP && lane == 0) {
        PROF_FLUSH(21, 25);
        PROF_FLUSH(27, 31);
    }
#endif
}

template <int D, bool KV8, int QT>
__global__ void __launch_bounds__(512, 1) msa_fwd_pipe_kernel(const __grid_constant__ FwdParams P)
{
    using C = PipeCfg<D, KV8, QT>;
    // The fp8 short-query variant multiplies in f16: code * 2^k as an f16 pair is two instructions per pair of codes (the bf16
    // image costs four) and exact for every legal scale, so Q, the arena blocks of a tile and P are f16 as well -- kind::f16
    // cannot mix the two formats in one MMA.  Q and the arena rows are converted as they are: what the variant asks of its
    // inputs (|q|, |arena k / v| <= 65504, include/msa.h) does not depend on the scales.
    constexpr bool F16 = KV8 && QT == 1;
    extern __shared__ __align__(1024) uint8_t smem[];
    const uint32_t sbase = smem_u32(smem);
    const uint32_t sQ = sbase, sRing = sbase + C::kQBytes;
    const uint32_t sStg = sRing + C::kRingBytes;
    (void)sStg;
    float2 *stats = reinterpret_cast<float2 *>(smem + C::kQBytes + C::kRingBytes + C::kStgBytes);
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem + C::kQBytes + C::kRingBytes + C::kStgBytes + C::kStatsBytes);
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(bars + kBarCount);
    const uint32_t bar0 = smem_u32(bars);
    auto bar = [bar0](int i) { return bar0 + static_cast<uint32_t>(i) * 8u; };

    const int warp = __shfl_sync(0xffffffffu, static_cast<int>(threadIdx.x >> 5), 0);
    const int lane = threadIdx.x & 31;
    if ((sbase & 1023u) != 0) __trap();

    // one-time setup: barriers, TMEM
    if (threadIdx.x == 0) {
        mbar_init(bar(kBarQFull), 1);
        mbar_init(bar(kBarQReady), kConvWarps);
        mbar_init(bar(kBarQEmpty), 1);
        for (int i = 0; i < C::kStages; ++i) {
            mbar_init(bar(kBarKvFull + i), F16 ? kConvWarps : KV8 ? 1 + kConvWarps : 1);  // the loader (+ KV8: every converter warp; f16: only they)
            mbar_init(bar(kBarKvDirect + i), 1);
            mbar_init(bar(kBarKvEmpty + i), kWritebackRing ? 2 : 1);   // the MMA warp's commit + the loader (or the write-back warp)
        }
        for (int i = 0; i < C::kStgStages; ++i) {
            mbar_init(bar(kBarStgFull + i), 1);
            mbar_init(bar(kBarStgEmpty + i), kConvWarps);
        }
        for (int c = 0; c < 2; ++c) {
            mbar_init(bar(kBarSFull + c), 1);
            mbar_init(bar(kBarPLo + c), 4);
            mbar_init(bar(kBarPQ2 + c), 4);
            mbar_init(bar(kBarPQ3 + c), 4);
            mbar_init(bar(kBarOFull + c), 1);
            mbar_init(bar(kBarOFree + c), 4);
            mbar_init(bar(kBarStFree + c), 4);
        }
        fence_mbar_init();
    }
    if (warp == 13) {
        tmem_alloc(smem_u32(tmem_slot), 512);
        tmem_relinquish();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    const int u_begin = P.cta_unit_begin[blockIdx.x], u_end = P.cta_unit_begin[blockIdx.x + 1];
    const int G = P.G, R = P.R;
    const float sl0 = P.scale_log2;

    if (warp < 8) {
        // =========================================================== softmax warpgroups
        asm volatile("setmaxnreg.inc.sync.aligned.u32 184;");
        const int c = warp >> 2;                       // chain
        const int row = threadIdx.x & 127;
        // row of a q tile -> token: token-major (row = t * G + g) or head-major (row = g * R + t), FwdParams::token_major
        const int t = P.token_major ? row / G : row % R;
        const uint32_t trow = tmem + (static_cast<uint32_t>((warp & 3) * 32) << 16);
        const uint32_t tS = trow + C::kColS + c * C::kChainCols;
        const uint32_t tO = trow + C::kColO + c * C::kChainCols;
        uint32_t ph_s = 0, ph_stfree = 1;
        PROF_DECL();
        for (int u = u_begin; u < u_end; ++u) {
            const WorkUnit wu = P.units[u];
            const int n = wu.tile_end - wu.tile_begin;
            if (n <= 0) continue;
            const bool pair = wu.mode == kModePair;
            const int steps = pair ? n : (n - c + 1) >> 1;
            if (steps <= 0) continue;
            const int p_row = wu.q_abs0 + (pair ? c * R : 0) + t;
            const int p_min = wu.q_abs0 + (pair ? c * R : 0);
            const float sl = sl0;
            // Token-major packing: the valid rows of the tile are its first tok * G rows.  A warp whose 32 rows lie beyond
            // them skips the unit's tiles altogether (its rows of S, P and O hold garbage nobody reads); the first warp of
            // the chain gives the idle warps' arrivals on the P barriers along with its own.
            uint32_t p_arrivals = 1;
            if (P.token_major) {
                const int tok = pair ? min(max(wu.n_tok - c * R, 0), R) : wu.n_tok;
                const int active = max(1, min(4, (tok * G + 31) >> 5));
                if ((warp & 3) >= active) {
                    ph_s ^= static_cast<uint32_t>(steps & 1);
                    mbar_wait(bar(kBarStFree + c), ph_stfree);
                    ph_stfree ^= 1;
                    stats[c * kTileM + row] = make_float2(0.f, 0.f);
                    // sync, not arrive: the warp stays here (in hardware, no issue slots) until the chain's working warps
                    // have finished the unit -- were it to go on and wait for S of the next unit, a barrier that is still
                    // several phases behind would show it the parity it expects
                    named_bar_sync(kNamedStFull + c, 256);
                    continue;
                }
                if ((warp & 3) == 0) p_arrivals += static_cast<uint32_t>(4 - active);
            }
            // Row state: integer reference `ref` (log2 units), l = sum of 2^(s*sl - ref) so far,
            // m_run = running max of the raw scores.  See msa_softmax.cuh.
            float ref = 0.f, l = 0.f, m_run = -INFINITY;
            bool has_ref = false;
            // Moves the reference up to ceil(m_run*sl) once it lags by more than the lazy
            // threshold: l and O (in TMEM) are multiplied by an exact power of two.  O may be
            // touched here because S of this tile is complete, hence so is PV of the last one.
            auto move_reference = [&](bool have_o) {
                const float tgt = (m_run == -INFINITY) ? ref : ceilf(m_run * sl);
                // a row that has seen no key yet (l = 0, O = 0) takes its first reference as is
                const bool first = !has_ref && m_run != -INFINITY;
                const bool grow = first || tgt - ref > C::kRescaleThreshold;
                if (__any_sync(0xffffffffu, grow)) {
                    const float alpha = (grow && !first) ? exp2_int(ref - tgt) : 1.f;
                    l *= alpha;
                    if (grow) ref = tgt;
                    has_ref = has_ref || first;
                    if (have_o) {
#pragma unroll
                        for (int q = 0; q < D / 16; ++q) {
                            uint32_t orr[16];
                            tmem_ld16(tO + q * 16, orr);
                            tmem_wait_ld();
#pragma unroll
                            for (int j = 0; j < 16; ++j) orr[j] = __float_as_uint(__uint_as_float(orr[j]) * alpha);
                            tmem_st16(tO + q * 16, orr);
                        }
                    }
                }
            };
            // tile summaries are fetched one tile ahead: the L2 round trip stays off the
            // P -> PV -> QK -> S critical loop of the chain
            const int2 *tip = reinterpret_cast<const int2 *>(P.tile_info + wu.tile_info_begin + wu.tile_begin + (pair ? 0 : c));
            const int ti_stride = pair ? 1 : 2;
            int2 ti_raw = __ldg(tip);
            for (int s = 0; s < steps; ++s) {
                const int tile = wu.tile_begin + (pair ? s : 2 * s + c);
                TileInfo ti;
                ti.max_abs = ti_raw.x;
                ti.ragged = ti_raw.y;
                if (s + 1 < steps) ti_raw = __ldg(tip + (s + 1) * ti_stride);
                const bool need_mask = ti.ragged != 0 || ti.max_abs > p_min;
                {
                    PROF_T0();
                    mbar_wait(bar(kBarSFull + c), ph_s);
                    PROF_ADD(0);
                }
                if ((threadIdx.x & 127) == 0) PROF_TRACE(1 + c, s, 0);
                ph_s ^= 1;
                tc_fence_after();
                PROF_T0();
                bool done = false;
                if (!need_mask && s > 0 && __all_sync(0xffffffffu, has_ref)) {
                    // fast path: stale reference, tile max found alongside, P handed over in parts
                    move_reference(true);
                    float tile_sum, tile_max;
                    done = softmax_fast_tile<F16>(tS, sl, ref, tile_sum, tile_max, [&](int part) {
                        __syncwarp();
                        if (lane == 0) mbar_arrive_n(bar((part == 0 ? kBarPLo : kBarPQ2) + c), p_arrivals);
                        if ((threadIdx.x & 127) == 0 && part == 0) PROF_TRACE(1 + c, s, 4);
                    }, [&](int ev) {
                        if ((threadIdx.x & 127) == 0) PROF_TRACE(1 + c, s, ev);
                    });
                    if (done) {
                        l += tile_sum;
                        m_run = fmaxf(m_run, tile_max);
                        __syncwarp();
                        if (lane == 0) mbar_arrive_n(bar(kBarPQ3 + c), p_arrivals);
                    }
                    PROF_ADD(20);
                }
                if (!done) {
                    // exact path (first tile of a unit, masked / ragged tiles, guard failures):
                    // all of S, mask, row max, reference moved BEFORE p is formed
                    uint32_t sr[128];
#pragma unroll
                    for (int q = 0; q < 4; ++q) tmem_ld32(tS + q * 32, *reinterpret_cast<uint32_t(*)[32]>(&sr[q * 32]));
                    tmem_wait_ld();
                    if (need_mask) {
                        const VBlock *vbp = P.vblocks + wu.vb_begin + tile * kVbPerTile;
#pragma unroll
                        for (int b = 0; b < kVbPerTile; ++b) {
                            const int4 e = __ldg(reinterpret_cast<const int4 *>(vbp + b));   // {src, abs_start, nvalid, paged}
                            int lim = min(e.z, p_row - e.y + 1);
                            if (tile * kVbPerTile + b >= wu.vb_count) lim = 0;               // past the causal horizon: not loaded
#pragma unroll
                            for (int j = 0; j < kBlock; ++j)
                                if (j >= lim) sr[b * kBlock + j] = 0xff800000u;             // -inf
                        }
                    }
                    float mx0 = -INFINITY, mx1 = -INFINITY;
#pragma unroll
                    for (int j = 0; j < 128; j += 4) {
                        mx0 = fmaxf(mx0, fmaxf(__uint_as_float(sr[j]), __uint_as_float(sr[j + 1])));
                        mx1 = fmaxf(mx1, fmaxf(__uint_as_float(sr[j + 2]), __uint_as_float(sr[j + 3])));
                    }
                    m_run = fmaxf(m_run, fmaxf(mx0, mx1));
                    move_reference(s > 0);
                    // p chunk by chunk, handed over in the same three parts as on the fast path: O += P V of the keys
                    // that are done runs while the rest is still being exponentiated
                    float sum0 = 0.f, sum1 = 0.f;
                    auto exact_chunk = [&](int q, uint32_t (&pk)[16]) {
#pragma unroll
                        for (int j = 0; j < 16; ++j) {
                            const float p0 = ex2_approx(fmaf(__uint_as_float(sr[q * 32 + 2 * j]), sl, -ref));
                            const float p1 = ex2_approx(fmaf(__uint_as_float(sr[q * 32 + 2 * j + 1]), sl, -ref));
                            sum0 += p0;
                            sum1 += p1;
                            pk[j] = F16 ? pack_f16x2(p0, p1) : pack_bf16x2(p0, p1);
                        }
                    };
                    auto publish = [&](int b) {
                        tc_fence_before();
                        __syncwarp();
                        if (lane == 0) mbar_arrive_n(bar(b + c), p_arrivals);
                    };
                    uint32_t pka[16], pkb[16];
                    exact_chunk(0, pka);
                    tmem_st16(tS, pka);
                    exact_chunk(1, pkb);
                    tmem_st16(tS + 16, pkb);
                    exact_chunk(2, pka);
                    tmem_wait_st_after(pka[12], pka[13], pka[14], pka[15]);
                    publish(kBarPLo);
                    tmem_st16(tS + 32, pka);
                    exact_chunk(3, pkb);
                    tmem_wait_st_after(pkb[12], pkb[13], pkb[14], pkb[15]);
                    publish(kBarPQ2);
                    tmem_st16(tS + 48, pkb);
                    l += sum0 + sum1;
                    tmem_wait_st();
                    publish(kBarPQ3);
                }
                PROF_ADD(2);
                if ((threadIdx.x & 127) == 0) PROF_TRACE(1 + c, s, 6);
                PROF_INC(4, 1);
                PROF_INC(6, done ? 1 : 0);
            }
            // hand (l, ref) of my row to the epilogue
            mbar_wait(bar(kBarStFree + c), ph_stfree);
            ph_stfree ^= 1;
            stats[c * kTileM + row] = make_float2(l, ref);
            named_bar_arrive(kNamedStFull + c, 256);
        }
#if defined(MSA_PROF) && MSA_PROF != 2
        if ((threadIdx.x & 127) == 0) {
            for (int i : {0, 2, 4, 6, 18, 20}) g_prof[blockIdx.x][i + c] += prof_acc[i];
        }
#endif
    } else if (warp < 12) {
        // =========================================================== epilogue warpgroup
        asm volatile("setmaxnreg.dec.sync.aligned.u32 80;");
        const int row = threadIdx.x & 127;
        const int t = P.token_major ? row / G : row % R;
        const int g = P.token_major ? row % G : row / R;
        const uint32_t trow = tmem + (static_cast<uint32_t>((warp & 3) * 32) << 16);
        uint32_t ph_o[2] = {0, 0};
        uint32_t cv_ent = 0, cv_stg = 0;       // KV8: ring entry / staging entry the converters are at (CTA-wide counters)
        uint32_t cv_phq = 0;                   // f16 variant: phase of the "Q landed" barrier the converters wait on
        uint32_t cv_dirpar = 0;                // f16 variant: per ring slot, parity of its "direct" barrier (used by some entries only)
        (void)cv_ent; (void)cv_stg; (void)cv_phq; (void)cv_dirpar;
        PROF_DECL();
        for (int u = u_begin; u < u_end; ++u) {
            const WorkUnit wu = P.units[u];
            const int n = wu.tile_end - wu.tile_begin;
            const bool pair = wu.mode == kModePair;
            const int rows_total = wu.n_tok * G;
            if constexpr (KV8) {
                // ---- converters (kv8_convert_unit): warp w of the four takes every fourth warp iteration of a tile
                kv8_convert_unit<C, D, F16>(P, wu, bar0, sQ, sStg, sRing, lane, 0x11111111u << (warp - 8), warp - 8, warp - 8, 4, cv_ent,
                                            cv_stg, cv_phq, cv_dirpar, blockIdx.x == 0 && u == u_begin && warp == 9 && lane == 0);
            }
            const int n_out = pair ? 2 : 1;                       // q tiles written by this unit
            for (int qt = 0; qt < n_out; ++qt) {
                const int tok = qt * R + t;
                const bool row_valid = (g < G) && (t < R) && (tok < wu.n_tok);
                const int head = row_valid ? P.kv_to_q[wu.kvh * G + g] : 0;
                float w0 = 0.f, w1 = 0.f, inv_l = 0.f, lse_val = -INFINITY;
                bool act0 = false, act1 = false;
                if (n > 0) {
                    // which chains hold (partial) results for this q tile
                    act0 = pair ? (qt == 0) : true;
                    act1 = pair ? (qt == 1) : (n >= 2);
                    float l0 = 0.f, m0 = -INFINITY, l1 = 0.f, m1 = -INFINITY;
                    if (act0) {
                        named_bar_sync(kNamedStFull + 0, 256);     // blocked in hardware until the chain's softmax warps are done
                        const float2 st = stats[0 * kTileM + row];
                        l0 = st.x;
                        m0 = st.y;
                        __syncwarp();
                        if (lane == 0) mbar_arrive(bar(kBarStFree + 0));
                    }
                    if (act1) {
                        named_bar_sync(kNamedStFull + 1, 256);     // blocked in hardware until the chain's softmax warps are done
                        const float2 st = stats[1 * kTileM + row];
                        l1 = st.x;
                        m1 = st.y;
                        __syncwarp();
                        if (lane == 0) mbar_arrive(bar(kBarStFree + 1));
                    }
                    // (l, ref) of each active chain; an inactive or empty chain weighs 0
                    const float mm = fmaxf((act0 && l0 > 0.f) ? m0 : -INFINITY, (act1 && l1 > 0.f) ? m1 : -INFINITY);
                    w0 = (act0 && l0 > 0.f) ? exp2_int(m0 - mm) : 0.f;
                    w1 = (act1 && l1 > 0.f) ? exp2_int(m1 - mm) : 0.f;
                    const float lt = w0 * l0 + w1 * l1;
                    if (lt > 0.f) {
                        inv_l = 1.f / lt;
                        lse_val = (mm + log2f(lt)) * 0.6931471805599453f;
                    }
                    w0 *= inv_l;
                    w1 *= inv_l;
                    if (act0) {
                        mbar_wait(bar(kBarOFull + 0), ph_o[0]);
                        ph_o[0] ^= 1;
                    }
                    if (act1) {
                        mbar_wait(bar(kBarOFull + 1), ph_o[1]);
                        ph_o[1] ^= 1;
                    }
                    tc_fence_after();
                }
                __nv_bfloat16 *orow = reinterpret_cast<__nv_bfloat16 *>(P.o) +
                                      (static_cast<size_t>(wu.q_row0 + tok) * P.Hq + head) * D;
                float *prow = P.workspace + (wu.partial_off < 0 ? 0 : wu.partial_off) +
                              static_cast<size_t>(g * wu.n_tok + tok) * D;
#pragma unroll
                for (int q = 0; q < D / 16; ++q) {
                    float acc[16];
#pragma unroll
                    for (int j = 0; j < 16; ++j) acc[j] = 0.f;
                    if (act0) {
                        uint32_t orr[16];
                        tmem_ld16(trow + C::kColO + q * 16, orr);
                        tmem_wait_ld();
#pragma unroll
                        for (int j = 0; j < 16; ++j) acc[j] = (w0 > 0.f) ? __uint_as_float(orr[j]) * w0 : 0.f;
                    }
                    if (act1) {
                        uint32_t orr[16];
                        tmem_ld16(trow + C::kColO + C::kChainCols + q * 16, orr);
                        tmem_wait_ld();
#pragma unroll
                        for (int j = 0; j < 16; ++j) acc[j] += (w1 > 0.f) ? __uint_as_float(orr[j]) * w1 : 0.f;
                    }
                    if (row_valid) {
                        if (wu.partial_off < 0) {
                            uint4 v0, v1;
                            v0.x = pack_bf16x2(acc[0], acc[1]);
                            v0.y = pack_bf16x2(acc[2], acc[3]);
                            v0.z = pack_bf16x2(acc[4], acc[5]);
                            v0.w = pack_bf16x2(acc[6], acc[7]);
                            v1.x = pack_bf16x2(acc[8], acc[9]);
                            v1.y = pack_bf16x2(acc[10], acc[11]);
                            v1.z = pack_bf16x2(acc[12], acc[13]);
                            v1.w = pack_bf16x2(acc[14], acc[15]);
                            *reinterpret_cast<uint4 *>(orow + q * 16) = v0;
                            *reinterpret_cast<uint4 *>(orow + q * 16 + 8) = v1;
                        } else {
#pragma unroll
                            for (int j = 0; j < 4; ++j)
                                *reinterpret_cast<float4 *>(prow + q * 16 + j * 4) =
                                    make_float4(acc[4 * j], acc[4 * j + 1], acc[4 * j + 2], acc[4 * j + 3]);
                        }
                    }
                }
                if (row_valid) {
                    if (wu.partial_off < 0)
                        P.lse[static_cast<size_t>(wu.q_row0 + tok) * P.Hq + head] = lse_val;
                    else
                        P.workspace[wu.partial_off + static_cast<size_t>(rows_total) * D + g * wu.n_tok + tok] = lse_val;
                }
                if (n > 0) {
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) {
                        if (act0) mbar_arrive(bar(kBarOFree + 0));
                        if (act1) mbar_arrive(bar(kBarOFree + 1));
                    }
                }
            }
        }
#if defined(MSA_PROF) && MSA_PROF != 2
#endif
    } else {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 64;");
        if (warp == 12 || warp == 14) {
            // ======================================================= loader warps (12: Q and K, 14: V)
            // Ring sequence: K of the CTA's i-th KV tile is entry 2i, its V entry 2i+1.
            const int which = warp == 12 ? 0 : 1;
            const CUtensorMap *tm_pool = which ? P.tm_pool_v : P.tm_pool_k;
            const CUtensorMap *tm_ctg = which ? P.tm_ctg_v : P.tm_ctg_k;
            const CUtensorMap *tm_ctg128 = which ? &P.tm_ctg_v128 : &P.tm_ctg_k128;
            RingPos rp{static_cast<uint32_t>(which), 1};
            // KV8: ring positions come from an entry counter (the ring order depends on the unit's mode), and this loader
            // also waits, in ring order, for the slots of the entries it does not fill: a waiter that does not see every
            // use of a slot cannot tell its barrier's phases apart (with few slots the V loader could otherwise run two
            // uses of a slot ahead of a V tile that is still being multiplied, find the parity it expects and overwrite it).
            uint32_t ent = 0;
            (void)ent;
            auto observe_until = [&](uint32_t target) {
                while (ent < target) {
                    mbar_wait(bar(kBarKvEmpty + (ent % C::kStages)), ((ent / C::kStages) & 1u) ^ 1u);
                    ++ent;
                }
            };
            uint32_t ph_qempty = 1;
            PROF_DECL();
            for (int u = u_begin; u < u_end; ++u) {
                const WorkUnit wu = P.units[u];
                const int n = wu.tile_end - wu.tile_begin;
                if (n <= 0) continue;
                if (which == 0) {
                    const int nq = wu.mode == kModePair ? 2 : 1;
                    mbar_wait(bar(kBarQEmpty), ph_qempty);
                    ph_qempty ^= 1;
                    if (P.token_major) {
                        // one box per q tile and 64-element half: G heads x R tokens, rows land as (token, head)
                        if (elect_one()) {
                            mbar_arrive_expect_tx(bar(kBarQFull), static_cast<uint32_t>(nq * G * R * D * 2));
                            const int hq0 = __ldg(P.kv_to_q + wu.kvh * G);
                            for (int c = 0; c < nq; ++c)
#pragma unroll
                                for (int h = 0; h < C::kHalves; ++h)
                                    tma_load_3d(sQ + c * C::kTileBytes + h * C::kHalfBytes, &P.tm_q3, bar(kBarQFull), h * 64, hq0,
                                                wu.q_row0 + c * R);
                        }
                    } else if (elect_one()) {
                        mbar_arrive_expect_tx(bar(kBarQFull), static_cast<uint32_t>(nq * G * R * D * 2));
                        for (int g = 0; g < G; ++g) {
                            const int hq = __ldg(P.kv_to_q + wu.kvh * G + g);
                            for (int c = 0; c < nq; ++c)
#pragma unroll
                                for (int h = 0; h < C::kHalves; ++h)
                                    tma_load_2d(sQ + c * C::kTileBytes + h * C::kHalfBytes + g * R * 128, &P.tm_q,
                                                bar(kBarQFull), hq * D + h * 64, wu.q_row0 + c * R);
                        }
                    }
                    __syncwarp();
                }
                const int c0 = wu.kvh * D;
                const uint32_t ent_base = ent;
                const bool pair_u = wu.mode == kModePair;
                (void)ent_base; (void)pair_u;
                // lane b < 8 owns virtual block b of a tile: fetch its entry, then resolve its row
                auto fetch = [&](int tile) -> int4 {
                    int4 e = make_int4(0, 0, 0, 0);
                    if (lane < kVbPerTile && tile < wu.tile_end && tile * kVbPerTile + lane < wu.vb_count)
                        e = __ldg(reinterpret_cast<const int4 *>(P.vblocks + wu.vb_begin + tile * kVbPerTile + lane));
                    return e;
                };
                auto resolve = [&](const int4 &e) -> ResolvedVb {
                    ResolvedVb r;
                    r.nvp = e.z | (e.w << 8);
                    if (KV8) r.row = e.x;                           // cached blocks come through the staging ring (warp 15)
                    else r.row = (e.z > 0 && e.w) ? __ldg(P.block_table + e.x) * kBlock : e.x;
                    return r;
                };
                // fused KV write-back: in a write-back launch warp 15 follows the ring, stores the arena blocks of
                // flagged units into their cache blocks straight from the ring slot, and gives every slot's second arrival
                const bool wb = P.vb_dst != nullptr;
                ResolvedVb cur = resolve(fetch(wu.tile_begin));
                ResolvedVb nxt = resolve(fetch(wu.tile_begin + 1));
                int4 raw = fetch(wu.tile_begin + 2);
#pragma unroll 1
                for (int j = 0; j < n; ++j) {
                    // One K (or V) tile into its ring slot, issued by one elected lane.  A full
                    // block is one 16-row box per 64-element half; eight full, consecutive arena
                    // blocks are one 128-row box; a partly filled block loads only its valid rows
                    // through the 8/4/2/1-row boxes: nothing outside a segment enters shared memory.
                    const int nv = cur.nvp & 0xff;
                    const uint32_t m_any = __ballot_sync(0xffffffffu, nv > 0) & 0xffu;
                    const uint32_t m_full = __ballot_sync(0xffffffffu, nv == kBlock) & 0xffu;
                    const uint32_t m_paged = __ballot_sync(0xffffffffu, (cur.nvp >> 8) != 0) & 0xffu;
                    const bool direct = !KV8 || (cur.nvp >> 8) == 0;          // this lane's block is loaded here, as bf16
                    const uint32_t m_dir = KV8 ? (m_any & ~m_paged) : m_any;
                    int rows_b[kVbPerTile];
#pragma unroll
                    for (int b = 0; b < kVbPerTile; ++b) rows_b[b] = __shfl_sync(0xffffffffu, cur.row, b);
                    const bool run = m_full == 0xffu && m_paged == 0 &&
                                     __all_sync(0xffffffffu, lane >= kVbPerTile || cur.row == rows_b[0] + lane * kBlock);
                    uint32_t slot = rp.slot, phase = rp.phase;
                    if constexpr (KV8) {
                        observe_until(ent_base + static_cast<uint32_t>(which ? kv8_entry_of_v(j, n, pair_u) : kv8_entry_of_k(j, pair_u)));
                        slot = ent % C::kStages;
                        phase = ((ent / C::kStages) & 1u) ^ 1u;
                        ++ent;
                    }
                    {
                        PROF_T0();
                        mbar_wait(bar(kBarKvEmpty + slot), phase);
                        PROF_ADD(16);
                    }
                    // f16 variant: the arena blocks land as bf16 and the converter warps rewrite them in place, so the loads (and
                    // this warp's zero fill) complete on the slot's "direct" barrier, every entry, and only the converters arrive on "full"
                    const uint32_t full = bar((F16 ? kBarKvDirect : kBarKvFull) + slot);
                    const uint32_t dst = sRing + slot * C::kTileBytes;
                    if (which == 1 && m_full != 0xffu) {
                        // V rows TMA will not write (block tails, blocks past the end / the horizon): zero them
                        // (generic-proxy stores, made visible to the tensor core's async proxy before the tile is armed)
#pragma unroll 1
                        for (int b = 0; b < kVbPerTile; ++b) {
                            const int nvb = __shfl_sync(0xffffffffu, nv, b);
                            const uint32_t off0 = static_cast<uint32_t>(nvb) * 128u;
#pragma unroll 1
                            for (int h = 0; h < C::kHalves; ++h)
                                for (uint32_t off = off0 + lane * 16u; off < kBlock * 128u; off += 512u)
                                    asm volatile("st.shared.v4.b32 [%0], {%1, %1, %1, %1};" ::"r"(dst + b * (kBlock * 128) + h * C::kHalfBytes + off), "r"(0u) : "memory");
                        }
                        fence_proxy_async_smem();
                        __syncwarp();
                    }
                    // f16 variant: an entry with neither arena blocks nor a zero fill does not use the "direct" barrier at all
                    // (the converter warps make the same test): no extra barrier hop on the common, all-cached tile
                    const bool skip_direct = F16 && m_dir == 0 && !(which == 1 && m_full != 0xffu);
                    if (skip_direct) {
                    } else if (run) {
                        if (elect_one()) {
                            mbar_arrive_expect_tx(full, static_cast<uint32_t>(kTileN * D * 2));
#pragma unroll
                            for (int h = 0; h < C::kHalves; ++h)
                                tma_load_2d(dst + h * C::kHalfBytes, tm_ctg128, full, c0 + h * 64, rows_b[0]);
                        }
                    } else if (m_any == m_full) {
                        if (elect_one()) {
                            mbar_arrive_expect_tx(full, static_cast<uint32_t>(__popc(m_dir) * kBlock * D * 2));
#pragma unroll
                            for (int b = 0; b < kVbPerTile; ++b) {
                                if (m_dir >> b & 1) {
                                    const CUtensorMap *tm = (m_paged >> b & 1) ? tm_pool : tm_ctg;
#pragma unroll
                                    for (int h = 0; h < C::kHalves; ++h)
                                        tma_load_2d(dst + b * (kBlock * 128) + h * C::kHalfBytes, tm, full, c0 + h * 64, rows_b[b]);
                                }
                            }
                        }
                    } else {
                        const uint32_t rows = __reduce_add_sync(0xffffffffu, static_cast<uint32_t>(direct ? nv : 0));
                        if (elect_one()) mbar_arrive_expect_tx(full, rows * D * 2);
                        __syncwarp();
                        if (nv > 0 && direct) {     // rare path: each lane issues the boxes of its own block
                            const CUtensorMap *tm = (cur.nvp >> 8) ? tm_pool : tm_ctg;
                            int off = 0;
#pragma unroll 1
                            for (int i = 0; i < 5; ++i) {
                                const int rows_i = kBlock >> i;
                                if (nv & rows_i) {
#pragma unroll 1
                                    for (int h = 0; h < C::kHalves; ++h)
                                        tma_load_2d(dst + lane * (kBlock * 128) + h * C::kHalfBytes + off * 128, tm + i, full,
                                                    c0 + h * 64, cur.row + off);
                                    off += rows_i;
                                }
                            }
                        }
                    }
                    __syncwarp();
                    // second arrival on the slot's empty barrier: here, at once, unless this is a write-back launch (then the
                    // write-back warp gives it for every tile, after its stores -- if any -- have read the slot)
                    if (kWritebackRing && !wb && elect_one()) mbar_arrive(bar(kBarKvEmpty + slot));
                    rp.advance2(C::kStages);
                    cur = nxt;
                    nxt = resolve(raw);
                    raw = fetch(wu.tile_begin + j + 3);
                }
                if constexpr (KV8) observe_until(ent_base + 2u * static_cast<uint32_t>(n));
            }
#if defined(MSA_PROF) && MSA_PROF != 2
            if (lane == 0) g_prof[blockIdx.x][16 + which] += prof_acc[16];
#endif
        } else if (warp == 13 && elect_one()) {
            // ======================================================= MMA issuer (one thread)
            constexpr uint32_t idesc_s = make_idesc(128, 128, false, F16);
            constexpr uint32_t idesc_o = make_idesc(128, D, true, F16);
            RingPos rk{0, 0}, rv{1, 0};
            uint32_t ph_q = 0, ph_p[2] = {0, 0}, ph_ofree[2] = {1, 1};
            int u = u_begin, tr_step = 0;    // (trace builds: which unit / KV step the issuer is in)
            (void)tr_step;
            PROF_DECL();
#if defined(MSA_PROF) && MSA_PROF != 2
            const long long prof_mma_start = clock64();
#endif
            uint32_t ment = 0;               // KV8: the ring is in the order of the take_k / take_v calls below
            (void)ment;
            auto take_k = [&]() -> uint32_t {
                if constexpr (KV8) {
                    const uint32_t slot = ment % C::kStages;
                    PROF_T0();
                    mbar_wait(bar(kBarKvFull + slot), (ment / C::kStages) & 1u);
                    PROF_ADD(8);
                    ++ment;
                    return slot;
                } else {
                    const uint32_t slot = rk.slot;
                    PROF_T0();
                    mbar_wait(bar(kBarKvFull + slot), rk.phase);
                    PROF_ADD(8);
                    rk.advance2(C::kStages);
                    return slot;
                }
            };
            auto take_v = [&]() -> uint32_t {
                if constexpr (KV8) {
                    const uint32_t slot = ment % C::kStages;
                    PROF_T0();
                    mbar_wait(bar(kBarKvFull + slot), (ment / C::kStages) & 1u);
                    PROF_ADD(9);
                    ++ment;
                    return slot;
                } else {
                    const uint32_t slot = rv.slot;
                    PROF_T0();
                    mbar_wait(bar(kBarKvFull + slot), rv.phase);
                    PROF_ADD(9);
                    rv.advance2(C::kStages);
                    return slot;
                }
            };
            // Descriptors: only the 14-bit start-address field (address >> 4) differs between the operands of one
            // tile, and it never carries out of its field (shared memory ends below 256 KB), so a tile's descriptor
            // is formed once and every MMA adds a compile-time constant to it: the issuing thread shares its SM
            // sub-partition with two softmax warps, and every instruction it does not need shortens the P -> S round trip.
            // (the high word -- SBO 1024, version, 128-byte swizzle -- is the same constant for all three operands)
            constexpr uint32_t kDescHi = make_smem_desc_hi(1024);
            const uint32_t q_desc = make_smem_desc_lo(sQ, 16);
            const uint32_t k_desc = make_smem_desc_lo(sRing, 16);
            const uint32_t v_desc = make_smem_desc_lo(sRing, C::kHalfBytes);
            constexpr uint32_t kTileStep = C::kTileBytes >> 4;
            auto qk = [&](int c, int qtile, uint32_t kslot) {
                const uint32_t qd = q_desc + qtile * kTileStep, kd = k_desc + kslot * kTileStep;
                const uint32_t d_tmem = tmem + C::kColS + c * C::kChainCols;
#pragma unroll
                for (int k = 0; k < D / 16; ++k) {
                    constexpr uint32_t kHalfStep = C::kHalfBytes >> 4;
                    const uint32_t off = (k >> 2) * kHalfStep + (k & 3) * 2;          // ((k>>2)*kHalfBytes + (k&3)*32) >> 4
                    umma_ss_lo<kDescHi>(d_tmem, qd + off, kd + off, idesc_s, k > 0);
                }
                umma_commit(bar(kBarSFull + c));
            };
            // O += P V in three parts: keys 0-63 as soon as the softmax warps have published the
            // first half of P, then keys 64-95 and 96-127 as they arrive.
            auto pv_lo = [&](int c, uint32_t vslot, bool first) {
                {
                    PROF_T0();
                    mbar_wait(bar(kBarPLo + c), ph_p[c]);
                    if (c == 0) PROF_ADD(10); else PROF_ADD(11);
                }
                if (first) {
                    PROF_T0();
                    mbar_wait(bar(kBarOFree + c), ph_ofree[c]);
                    PROF_ADD(12);
                    ph_ofree[c] ^= 1;
                }
                tc_fence_after();
                const uint32_t vd = v_desc + vslot * kTileStep;
#pragma unroll
                for (int k = 0; k < kTileN / 32; ++k)
                    umma_ts_lo<kDescHi>(tmem + C::kColO + c * C::kChainCols, tmem + C::kColS + c * C::kChainCols + k * 8,
                            vd + k * ((kBlock * 128) >> 4), idesc_o, (!first || k > 0) ? 1u : 0u);
            };
            auto pv_hi = [&](int c, uint32_t vslot) {
                const uint32_t vd = v_desc + vslot * kTileStep;
                mbar_wait(bar(kBarPQ2 + c), ph_p[c]);
                PROF_TRACE(0, tr_step, 7 + 2 * c);
                tc_fence_after();
#pragma unroll
                for (int k = kTileN / 32; k < 3 * kTileN / 64; ++k)
                    umma_ts_lo<kDescHi>(tmem + C::kColO + c * C::kChainCols, tmem + C::kColS + c * C::kChainCols + k * 8,
                            vd + k * ((kBlock * 128) >> 4), idesc_o, 1u);
                mbar_wait(bar(kBarPQ3 + c), ph_p[c]);
                PROF_TRACE(0, tr_step, 8 + 2 * c);
                ph_p[c] ^= 1;
                tc_fence_after();
#pragma unroll
                for (int k = 3 * kTileN / 64; k < kTileN / 16; ++k)
                    umma_ts_lo<kDescHi>(tmem + C::kColO + c * C::kChainCols, tmem + C::kColS + c * C::kChainCols + k * 8,
                            vd + k * ((kBlock * 128) >> 4), idesc_o, 1u);
            };
            auto pv = [&](int c, uint32_t vslot, bool first) {
                pv_lo(c, vslot, first);
                pv_hi(c, vslot);
            };
            for (u = u_begin; u < u_end; ++u) {
                const WorkUnit wu = P.units[u];
                const int n = wu.tile_end - wu.tile_begin;
                if (n <= 0) continue;
                {
                    PROF_T0();
                    mbar_wait(bar(F16 ? kBarQReady : kBarQFull), ph_q);
                    PROF_ADD(13);
                }
                ph_q ^= 1;
                if (wu.mode == kModePair) {
                    uint32_t ks = take_k();
                    tc_fence_after();
                    qk(0, 0, ks);
                    qk(1, 1, ks);
                    umma_commit(bar(kBarKvEmpty + ks));
                    if (n == 1) umma_commit(bar(kBarQEmpty));
                    for (int j = 0; j < n; ++j) {
                        tr_step = j;
                        PROF_TRACE(0, j, 0);
                        const uint32_t vs = take_v();
                        PROF_TRACE(0, j, 1);
                        // the K tile of the next step is taken while the second half of P is still
                        // being formed, so QK follows PV without a barrier round trip in between
                        pv_lo(0, vs, j == 0);
                        if (j + 1 < n) {
                            ks = take_k();
                            tc_fence_after();
                        }
                        pv_hi(0, vs);
                        PROF_TRACE(0, j, 2);
                        if (j == n - 1) umma_commit(bar(kBarOFull + 0));
                        if (j + 1 < n) {
                            PROF_TRACE(0, j, 3);
                            qk(0, 0, ks);
                            PROF_TRACE(0, j, 4);
                        }
                        pv(1, vs, j == 0);
                        PROF_TRACE(0, j, 5);
                        umma_commit(bar(kBarKvEmpty + vs));
                        if (j == n - 1) umma_commit(bar(kBarOFull + 1));
                        if (j + 1 < n) {
                            qk(1, 1, ks);
                            PROF_TRACE(0, j, 6);
                            umma_commit(bar(kBarKvEmpty + ks));
                            if (j + 2 == n) umma_commit(bar(kBarQEmpty));
                        }
                    }
                } else {
                    uint32_t ks = take_k();
                    tc_fence_after();
                    qk(0, 0, ks);
                    umma_commit(bar(kBarKvEmpty + ks));
                    if (n > 1) {
                        ks = take_k();
                        tc_fence_after();
                        qk(1, 0, ks);
                        umma_commit(bar(kBarKvEmpty + ks));
                    }
                    if (n <= 2) umma_commit(bar(kBarQEmpty));
                    for (int j = 0; j < n; ++j) {
                        const int c = j & 1;
                        tr_step = j;
                        PROF_TRACE(0, j, 0);
                        const uint32_t vs = take_v();
                        PROF_TRACE(0, j, 1);
                        pv(c, vs, j < 2);
                        PROF_TRACE(0, j, 2);
                        umma_commit(bar(kBarKvEmpty + vs));
                        if (j + 2 >= n) umma_commit(bar(kBarOFull + c));
                        if (j + 2 < n) {
                            ks = take_k();
                            PROF_TRACE(0, j, 3);
                            tc_fence_after();
                            qk(c, 0, ks);
                            PROF_TRACE(0, j, 4);
                            umma_commit(bar(kBarKvEmpty + ks));
                            if (j + 3 == n) umma_commit(bar(kBarQEmpty));
                        }
                    }
                }
            }
#if defined(MSA_PROF) && MSA_PROF != 2
            prof_acc[14] = static_cast<unsigned long long>(clock64() - prof_mma_start);
            PROF_FLUSH(8, 15);
#endif
        }
        else if (KV8 && warp == 15) {
            // ======================================================= KV8: loader of the fp8 blocks (staging ring)
            // Ring entries in ring order; for every entry whose tile holds cached blocks, their codes go into the next
            // staging slot (block b at b * 16 * D, rows of D bytes, no swizzle).  Independent of the bf16 ring, so the fp8
            // stream runs kStgStages entries ahead of the converters whatever the tensor core is doing.
            uint32_t stg = 0;
            PROF_DECL();
#if defined(MSA_PROF) && MSA_PROF != 2
            const long long prof_stg_start = clock64();
#endif
            for (int u = u_begin; u < u_end; ++u) {
                const WorkUnit wu = P.units[u];
                const int n = wu.tile_end - wu.tile_begin;
                if (n <= 0) continue;
                const int c0 = wu.kvh * D;
                const bool pair_u = wu.mode == kModePair;
                auto fetch = [&](int e) -> int4 {                 // vblock entry of lane b < 8 for ring entry e (zeros past the unit)
                    int4 v = make_int4(0, 0, 0, 0);
                    if (e < 2 * n) {
                        bool is_v;
                        int t;
                        kv8_entry(e, n, pair_u, is_v, t);
                        const int tile = wu.tile_begin + t;
                        if (lane < kVbPerTile && tile * kVbPerTile + lane < wu.vb_count)
                            v = __ldg(reinterpret_cast<const int4 *>(P.vblocks + wu.vb_begin + tile * kVbPerTile + lane));
                    }
                    return v;
                };
                auto resolve = [&](const int4 &v) -> ResolvedVb {     // nvp = valid slots of a CACHED block (0 otherwise)
                    ResolvedVb r;
                    const bool pg = v.z > 0 && v.w != 0;
                    r.nvp = pg ? v.z : 0;
                    r.row = pg ? __ldg(P.block_table + v.x) * kBlock : 0;
                    return r;
                };
                ResolvedVb cur = resolve(fetch(0));
                ResolvedVb nxt = resolve(fetch(1));
                int4 raw = fetch(2);
#pragma unroll 1
                for (int e = 0; e < 2 * n; ++e) {
                    const int nv = cur.nvp;
                    const uint32_t m_paged = __ballot_sync(0xffffffffu, nv > 0) & 0xffu;
                    const uint32_t m_full = __ballot_sync(0xffffffffu, nv == kBlock) & 0xffu;
                    if (m_paged != 0) {
                        bool is_v;
                        int t;
                        kv8_entry(e, n, pair_u, is_v, t);
                        const CUtensorMap *tm = is_v ? P.tm_pool_v : P.tm_pool_k;
                        const uint32_t st = stg % static_cast<uint32_t>(C::kStgDiv);
                        const uint32_t rows = __reduce_add_sync(0xffffffffu, static_cast<uint32_t>(nv));
                        {
                            PROF_T0();
                            mbar_wait(bar(kBarStgEmpty + st), ((stg / C::kStgDiv) & 1u) ^ 1u);
                            PROF_ADD(25);
                        }
                        const uint32_t full = bar(kBarStgFull + st);
                        const uint32_t dst = sStg + st * C::kStgTileBytes;
                        if (m_paged == m_full) {
                            int rows_b[kVbPerTile];
#pragma unroll
                            for (int b = 0; b < kVbPerTile; ++b) rows_b[b] = __shfl_sync(0xffffffffu, cur.row, b);
                            if (elect_one()) {
                                mbar_arrive_expect_tx(full, rows * D);
#pragma unroll
                                for (int b = 0; b < kVbPerTile; ++b)
                                    if (m_paged >> b & 1) tma_load_2d(dst + b * (kBlock * D), tm, full, c0, rows_b[b]);
                            }
                        } else {
                            if (elect_one()) mbar_arrive_expect_tx(full, rows * D);
                            __syncwarp();
                            if (nv > 0) {     // a partly filled block loads only its valid rows (8/4/2/1-row boxes)
                                int off = 0;
#pragma unroll 1
                                for (int i = 0; i < 5; ++i) {
                                    const int rows_i = kBlock >> i;
                                    if (nv & rows_i) {
                                        tma_load_2d(dst + lane * (kBlock * D) + off * D, tm + i, full, c0, cur.row + off);
                                        off += rows_i;
                                    }
                                }
                            }
                        }
                        __syncwarp();
                        ++stg;
                    }
                    cur = nxt;
                    nxt = resolve(raw);
                    raw = fetch(e + 3);
                }
            }
#if defined(MSA_PROF) && MSA_PROF != 2
            prof_acc[26] = static_cast<unsigned long long>(clock64() - prof_stg_start);
            if (lane == 0) PROF_FLUSH(25, 27);
#endif
        }
        else if (warp == 15 && P.vb_dst != nullptr) {
            // ======================================================= write-back warp (plans from msa_plan_create_writeback)
            // Follows the ring like the MMA warp.  In a flagged unit, once a K or V tile has landed, lane b stores virtual
            // block b -- if it is an arena block with a destination -- into the cache (one TMA store per 64-element half,
            // same box and swizzle as the load, partly filled blocks through the 8/4/2/1-row boxes), and when the stores
            // have read the slot the warp gives the slot's second "empty" arrival that the loader gives everywhere else.
            uint32_t entry = 0;                              // ring entry of K of the CTA's next tile (V: entry + 1)
            int held = -1;                                   // slot whose stores may still be reading it (released one entry later)
            for (int u = u_begin; u < u_end; ++u) {
                const WorkUnit wu = P.units[u];
                const int n = wu.tile_end - wu.tile_begin;
                if (n <= 0) continue;
                const int c0 = wu.kvh * D;
#pragma unroll 1
                for (int j = 0; j < n; ++j) {
                    const int tile = wu.tile_begin + j;
                    int dsti = -1, nv = 0, drow = 0;
                    // is this tile mine to store?  (the planner deals the tiles out among the units that load them)
                    if (wu.writeback != 0 && __ldg(P.tile_writer + wu.tile_info_begin + tile) == wu.q_row0 && lane < kVbPerTile &&
                        tile * kVbPerTile + lane < wu.vb_count) {
                        const int idx = wu.vb_begin + tile * kVbPerTile + lane;
                        const int4 e = __ldg(reinterpret_cast<const int4 *>(P.vblocks + idx));   // {src, abs_start, nvalid, paged}
                        if (e.z > 0 && e.w == 0) {
                            dsti = __ldg(P.vb_dst + idx);
                            nv = e.z;
                            if (dsti >= 0) drow = __ldg(P.block_table + dsti) * kBlock;
                        }
                    }
                    const bool stores = __any_sync(0xffffffffu, dsti >= 0);
#pragma unroll 1
                    for (int which = 0; which < 2; ++which, ++entry) {
                        const uint32_t slot = entry % C::kStages, parity = (entry / C::kStages) & 1u;
                        const CUtensorMap *tm_pool = which ? P.tm_pool_v : P.tm_pool_k;
                        // Every tile of every unit, in ring order: a waiter that skips ahead (or is lapped) by two uses of a slot
                        // cannot tell the phases apart, and an arrival given before the loader has taken the slot for THIS tile
                        // would count for the slot's previous use and hand it back while the MMAs still read it.
                        mbar_wait(bar(kBarKvFull + slot), parity);
                        if (stores) {
                            if (dsti >= 0) {
                                const uint32_t src = sRing + slot * C::kTileBytes + lane * (kBlock * 128);
                                int off = 0;
#pragma unroll 1
                                for (int i = 0; i < 5; ++i) {
                                    const int rows_i = kBlock >> i;
                                    if (nv & rows_i) {
#pragma unroll 1
                                        for (int h = 0; h < C::kHalves; ++h)
                                            tma_store_2d(tm_pool + i, src + h * C::kHalfBytes + off * 128, c0 + h * 64, drow + off);
                                        off += rows_i;
                                    }
                                }
                            }
                            tma_store_commit();                      // (an empty group for lanes without a block)
                            if (held >= 0) {                         // the group before this one has read its slot by now
                                asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory");
                                __syncwarp();
                                if (lane == 0) mbar_arrive(bar(kBarKvEmpty + held));
                            }
                            held = static_cast<int>(slot);
                        } else {
                            if (held >= 0) {
                                tma_store_wait_read();
                                __syncwarp();
                                if (lane == 0) mbar_arrive(bar(kBarKvEmpty + held));
                                held = -1;
                            }
                            if (lane == 0) mbar_arrive(bar(kBarKvEmpty + slot));
                        }
                    }
                }
            }
            if (held >= 0) {
                tma_store_wait_read();
                __syncwarp();
                if (lane == 0) mbar_arrive(bar(kBarKvEmpty + held));
            }
            tma_store_wait_all();                            // the data is in global memory before the CTA retires
        }
#if defined(MSA_PROF) && MSA_PROF == 2
        else if (warp == 15 && lane == 0 && blockIdx.x == 0 && u_begin < u_end) {
            // observer (trace builds only): when does each chain's S become complete in the first unit?
            const WorkUnit wu = P.units[u_begin];
            const int n = wu.tile_end - wu.tile_begin;
            if (wu.mode == kModePair) {
                uint32_t ph = 0;
                for (int s = 0; s < n && s < 64; ++s) {
                    mbar_wait(bar(kBarSFull + 0), ph);
                    g_trace[3][s][0] = clock64();
                    mbar_wait(bar(kBarSFull + 1), ph);
                    g_trace[3][s][1] = clock64();
                    ph ^= 1;
                }
            }
        }
#endif
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 13) tmem_dealloc(tmem, 512);
}

}  // namespace msa
