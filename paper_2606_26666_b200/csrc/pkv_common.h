// pkv_common.h -- internal declarations shared by the host planner and the CUDA translation
// units of libpkv.  Not part of the ABI (include/pkv.h is).
#pragma once

#include <cstddef>
#include <cstdint>

#include "pkv.h"

namespace pkv {

constexpr int kD = 128;         // head dimension compiled in
constexpr int kBlock = 16;      // tokens per K/V stage (one TMA box); pages hold 1, 2 or 4 blocks
constexpr int kAutoCMin = 4;    // PAPER.md:85 "C_min = 4 CTAs/SM" (auto split rule, A12)
constexpr int kMaxSplits = 256; // cap on S (and on n_i in FIXED_CHUNK mode)
constexpr int kAllFlags = PKV_FLAG_VALIDATE | PKV_FLAG_NO_PDL | PKV_FLAG_SEPARATE_BUILD | PKV_FLAG_TEST_REPLAN | PKV_FLAG_OUT_PINNED;
constexpr int kDefaultPrefetchKb = 256;   // policy.prefetch_kb == 0
constexpr int kMaxFusedRows = 512;  // fused build (TMA kernel): the batch's offsets and lengths sit in shared memory

void set_error(const char* fmt, ...);
void clear_error();

inline int64_t ceil_div64(int64_t a, int64_t b) { return (a + b - 1) / b; }
inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// Device-resident header at the front of the workspace (and of the host-planned queue image).
// Written by the builder kernel (or by the host planner), read by decode / merge / counters.
struct QueueHeader {
    int32_t num_tasks;       // entries in the task list (rect route: includes empty intervals)
    int32_t max_row_splits;  // max_i n_i (rect: S)
    int32_t total_row_slots; // split_offsets[B]
    int32_t resolved_splits; // S
    int32_t empty_tasks;     // rect route: entries with t_begin >= t_end
    int32_t work_counter;    // dynamic task scheduler; self-resetting
    int32_t done_counter;    // CTAs that finished; self-resetting
    int32_t error_word;      // pkv_device_error bits; sticky (kernels only ever OR into it)
    int64_t sum_seq_lens;    // sum_i N_i
    int32_t build_launches;  // 1: written by the builder kernel, 0: by the decode kernel's fused build / the host
    int32_t chunk_tiles;     // FIXED_CHUNK / BALANCED: resolved tiles per task, else 0
    int32_t launched_build;  // what the last build / decode on this workspace really launched:
    int32_t launched_decode; //   every kernel leaves its mark (pkv_counters.launched_*)
    int32_t launched_merge;
    int32_t pad_;
};
static_assert(sizeof(QueueHeader) == 64, "QueueHeader layout");

// One (row, split) pair of the queue: what a work unit of the TMA kernel needs, in one 32-byte
// load (the Hkv tasks of the pair share it; task(i, g, s) sits at so*Hkv + g*n + s).  Private.
struct RowSlot {
    int32_t row;
    int32_t so;     // split_offsets[row]
    int32_t n;      // slots of the row (n_i, or S on the rect route)
    int32_t split;
    int32_t tok0;   // token range [tok0, tok1) -- empty when tok0 >= tok1
    int32_t tok1;
    int32_t grow;   // request row (= row unless the launch is indexed, pkv_decode_indexed)
    int32_t nlen;   // the row's length N_i (the fused KV-append needs the position of its last token)
};
static_assert(sizeof(RowSlot) == 32, "RowSlot layout");

// Policy with every "0 = auto" field resolved.
struct Resolved {
    int32_t S;          // split count (FIXED_COUNT) or cap on n_i (FIXED_CHUNK)
    int32_t tile_tokens;
    int32_t split_mode;
    int32_t chunk_tiles;
    int32_t route;
    int32_t merge_mode;
    int32_t kernel;
    int32_t G;
    int32_t num_sms;    // BALANCED: U (policy.num_sms, else the device's)
    int32_t flags;      // pkv_flag bits
    int32_t heads_per_cta;  // 0 = automatic
    int32_t prefetch_kb;    // resolved: 0 = off
    int32_t auto_mode;      // policy said PKV_SPLIT_AUTO (resolved to BALANCED here; pkv_decode_host re-plans per step)
};

// Byte offsets inside the caller's workspace.  Pure function of (shape, S bound).
struct WorkspaceLayout {
    size_t header, fuse_counters, init_bytes, split_offsets, rowslots, tasks, part_m, part_l, part_acc, total;
    int64_t slots_cap; // B * Hkv * S
};

// Validates shape/policy (host-checkable part).  num_sms_or_0: SM count to use when the policy
// says num_sms == 0 and num_splits == 0; if that is 0 too, S resolves to kMaxSplits when
// `bound_ok`, else an error is returned.
pkv_status validate_and_resolve(const pkv_shape* shape, const pkv_split_policy* policy,
                                int num_sms_or_0, bool bound_ok, Resolved* out);
WorkspaceLayout workspace_layout(const pkv_shape& shape, int32_t S);

// Row-local split bounds (A6): T tiles, c tiles per split, n non-empty
// splits.  Same integer formulas on host and device.
struct RowSplits { int32_t T, c, n; };
#if defined(__CUDACC__)
__host__ __device__
#endif
inline RowSplits row_splits(int32_t N, int32_t tile_tokens, int32_t split_mode, int32_t S,
                            int32_t chunk_tiles) {
    RowSplits r;
    r.T = N > 0 ? (N + tile_tokens - 1) / tile_tokens : 0;
    if (r.T == 0) { r.c = 0; r.n = 0; return r; }
    int32_t Si = S;
    if (split_mode != PKV_SPLIT_FIXED_COUNT) {   // FIXED_CHUNK, or BALANCED with its chunk resolved
        int32_t want = (r.T + chunk_tiles - 1) / chunk_tiles;
        Si = want < S ? want : S;
    }
    r.c = (r.T + Si - 1) / Si;
    r.n = (r.T + r.c - 1) / r.c;
    return r;
}

// BALANCED split mode (include/pkv.h; A21): the batch-wide chunk, from W = sum_i T_i,
// U = num_sms and `fits(c)` = [sum_i ceil(T_i / c) <= U] (monotone in c).  The caller supplies
// fits; host and device search the same interval the same way.
constexpr int kBalWaves = 32;        // many-wave regime: about 32 pairs per SM
constexpr int kBalMinTokens = 256;   // ... of at least 256 tokens each
template <typename Fits>
#if defined(__CUDACC__)
__host__ __device__
#endif
inline int32_t balanced_chunk(int64_t W, int32_t U, int32_t tile_tokens, Fits fits) {
    if (W <= 0 || U <= 0) return 1;
    const int64_t m = (kBalMinTokens + tile_tokens - 1) / tile_tokens;
    const int64_t w = (W + (int64_t)kBalWaves * U - 1) / ((int64_t)kBalWaves * U);
    const int64_t c2 = w > m ? w : m;            // many-wave chunk
    int64_t lo = (W + U - 1) / U, hi = lo + c2;  // single wave: c in [ceil(W/U), ceil(W/U) + c2]
    if (fits((int32_t)hi)) {
        while (lo < hi) {   // smallest c in [lo, hi] that fits
            const int64_t mid = (lo + hi) >> 1;
            if (fits((int32_t)mid)) hi = mid; else lo = mid + 1;
        }
        return (int32_t)lo;
    }
    return (int32_t)c2;
}

// KV heads one CTA of the TMA kernel streams together: the largest divisor of Hkv in {8, 4, 2, 1}
// that still leaves work units for at least 85 % of the SMs (units = row slots x Hkv / HG; whole-page
// boxes stream faster than head slices, so 128 units of two heads beat 256 units of one on 148 SMs:
// config 2, S = 32: 23.4 vs 24.2 us per step).
// max_hg: 4 when G = 16 (two warps per KV head, one per block of 8 query heads) or d = 256 (a stage
// of 8 heads would be 128 KiB), else 8.
inline int max_heads_per_cta(int G, int d) { return (G == 16 || d == 256) ? 4 : 8; }
inline int choose_heads_per_cta(int forced, int Hkv, int64_t row_slots, int num_sms, int max_hg = 8) {
    if (forced > 0 && Hkv % forced == 0 && forced <= max_hg) return forced;
    int best = 1;
    for (int hg = max_hg; hg >= 1; hg >>= 1) {
        if (hg > Hkv || Hkv % hg) continue;
        best = hg;
        if (row_slots * (Hkv / hg) * 20 >= (int64_t)num_sms * 17) return hg;
    }
    return best;   // nothing fills the machine: smallest valid group = most units
}

// Host planner shared by pkv_build_workqueue_host and pkv_decode_host.
pkv_status plan_host(const pkv_shape& shape, const Resolved& rp, const int32_t* seq_lens,
                     pkv_task* tasks, int32_t tasks_cap, int32_t* split_offsets, RowSlot* rowslots,
                     QueueHeader* hdr, int32_t* max_unit_tokens = nullptr);

// Cost-model constants fitted on B200: read probe, the cost of one more
// dependent kernel in a replayed step, work items per SM that saturate the read rate.
constexpr double kB200BetaGbps = 7060.0;
constexpr double kB200LambdaUs = 2.0;
constexpr double kB200CMin = 0.72;
// A27: streaming efficiency of a CTA that reads HG heads' slices of every page (HG * d * 2 bytes
// per token row out of Hkv * d * 2): whole pages stream at beta, single-head slices at 0.87 beta
// (config 2, decode kernel alone: 20.5 / 21.4 / 21.8 / 23.5 us at HG = 8 / 4 / 2 / 1).
inline double head_slice_efficiency(int hg) { return hg >= 8 ? 1.0 : (hg >= 4 ? 0.96 : (hg >= 2 ? 0.94 : 0.87)); }

}  // namespace pkv
