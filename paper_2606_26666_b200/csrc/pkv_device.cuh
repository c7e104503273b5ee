// pkv_device.cuh -- device-side declarations shared by the CUDA translation units of libpkv:
// kernel parameter block, PTX wrappers (mbarrier, TMA, ldmatrix, HMMA), and the task epilogue
// (partial-state store, direct output, fused merge) used by both decode kernels.
#pragma once

#include <cuda_fp16.h>
#include <cuda_runtime.h>

#include <utility>

#include "pkv_common.h"

namespace pkv {

constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;

struct PlanArgs {   // split policy as the device-side planner needs it
    int32_t B, Hkv, S, tile_tokens, split_mode, chunk_tiles, route, num_sms;
    int32_t flags;        // pkv_flag bits
    int32_t max_tokens;   // max_pages * page_size: the longest row the block table can describe
    const int32_t* row_index;   // indexed rows (pkv_decode_indexed): launch row i is request row_index[i]; or nullptr
};

// Request row of launch row i: the row of q, out, lse, block_table and seq_lens it works on.
__device__ __forceinline__ int32_t request_row(const int32_t* row_index, int i) {
    return row_index ? __ldcg(row_index + i) : i;
}

struct DecodeParams {
    const __half* q;            // [B, Hq, d]
    const __half* k_cache;      // raw pointers (SIMT kernel; the TMA kernel uses tensor maps)
    const __half* v_cache;
    const int32_t* block_table; // [B, max_pages]
    const int32_t* seq_lens;    // [B]
    const int32_t* row_index;   // [B] or nullptr: launch row -> request row (q, out, lse, block_table, seq_lens)
    pkv_task* tasks;              // written by the builder / the fused build, read by the SIMT kernel
    RowSlot* rowslots;            // [split_offsets[B]] (row, split) pairs
    int32_t* split_offsets;       // [B+1]
    QueueHeader* hdr;
    __half* out;                // [B, Hq, d]
    float* lse;                 // [B, Hq] or nullptr
    float* part_m;              // [slots, G]
    float* part_l;              // [slots, G]
    float* part_acc;            // [slots, G, d]
    int32_t* fuse_counters;     // [B*Hkv]
    int64_t stride_page, stride_token, stride_head; // elements
    int32_t B, Hq, Hkv, max_pages, tile_tokens, merge_mode;
    int32_t d;                   // head dimension: 64, 128 or 256
    const float* k_scale;        // FP8 caches: per-KV-head scales [Hkv] or nullptr (= 1)
    const float* v_scale;
    // fused KV-append (+RoPE) before decode (pkv_decode_append; reading A29), or nullptr
    const __half* k_new;         // [rows, Hkv, d]: the new token's K (before RoPE), by request row
    const __half* v_new;         // [rows, Hkv, d]
    const float* rope_cos;       // [rope_positions, d/2] or nullptr (no rotation)
    const float* rope_sin;
    int32_t rope_positions;
    PlanArgs plan;               // split policy (fused build)
    int64_t tasks_cap;
    int32_t fused_build;         // TMA kernel: 1 = every CTA derives the queue from seq_lens itself
    int32_t heads_per_cta;       // TMA kernel: KV heads one CTA streams together (1, 2, 4 or 8)
    int32_t dynamic_sched;      // 1: tasks handed out by an atomic counter
    int32_t force_replan;       // test hook: treat the speculative plan as invalidated
    int32_t prefetch_pages;     // TMA kernel: 16-token blocks of its first unit a CTA prefetches into L2 before the wait
    int32_t page_shift;         // log2(page_size / 16): a page holds 1, 2 or 4 blocks of 16 tokens
    float scale;                // x = scale * <q, k>
    float scale_log2;           // scale * log2(e)
    int64_t num_pages;          // PKV_FLAG_VALIDATE: block-table entries must lie in [0, num_pages)
#ifdef PKV_TRACE
    unsigned long long* trace;  // trace build only: [grid][16] %globaltimer stamps, or nullptr
#endif
};

// ------------------------------------------------------------------ small PTX wrappers

__device__ __forceinline__ float ex2_approx(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void sts_b32(uint32_t addr, uint32_t v) {
    asm volatile("st.shared.b32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}
__device__ __forceinline__ void named_bar_arrive(int id, int nthreads) {
    asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}
__device__ __forceinline__ void named_bar_sync(int id, int nthreads) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// Programmatic dependent launch (PDL): every kernel of the step lets its successor's CTAs be
// scheduled early and waits for its predecessor's results before touching global memory.
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// Phase stamps (%globaltimer) for the step timeline: compiled in only with -DPKV_TRACE (a separate
// trace build of the library); the release build carries no stamp, no pointer and no hook.
#ifdef PKV_TRACE
__device__ __forceinline__ void trace_stamp(const DecodeParams& p, int slot) {
    if (p.trace) {
        unsigned long long t;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
        p.trace[(size_t)blockIdx.x * 16 + slot] = t;
    }
}
// the merge kernel's CTA 0 stamps row kTraceMergeRow of the same buffer
constexpr int kTraceMergeRow = 148;
__device__ __forceinline__ void trace_stamp_row(const DecodeParams& p, int row, int slot) {
    if (p.trace) {
        unsigned long long t;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
        p.trace[(size_t)row * 16 + slot] = t;
    }
}
#define PKV_TRACE_STAMP(p, slot) trace_stamp(p, slot)
#define PKV_TRACE_STAMP_MERGE(p, slot) trace_stamp_row(p, kTraceMergeRow, slot)
#else
#define PKV_TRACE_STAMP(p, slot) ((void)0)
#define PKV_TRACE_STAMP_MERGE(p, slot) ((void)0)
#endif

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    while (!mbar_try_wait(bar, parity)) {
    }
}

// TMA tile loads (cp.async.bulk.tensor), completion on an mbarrier of this CTA.
// `policy`: an L2 cache policy (l2_policy_evict_first): the K/V stream is read once per step, so
// its lines are the first to go and the step's small, re-read data (seq_lens, block table, q,
// split_offsets, partial states) stays in L2 across the 100+ MB that stream through it.
__device__ __forceinline__ void tma_load_5d(uint32_t dst, const void* tmap, uint32_t bar, int c0, int c1,
                                            int c2, int c3, int c4, unsigned long long policy) {
    asm volatile(
        "cp.async.bulk.tensor.5d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint "
        "[%0], [%1, {%3, %4, %5, %6, %7}], [%2], %8;" ::"r"(dst),
        "l"(tmap), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4), "l"(policy)
        : "memory");
}
__device__ __forceinline__ unsigned long long l2_policy_evict_first() {
    unsigned long long pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
// L2 prefetch of one tensor-map box (no shared-memory destination, no completion): used BEFORE the
// kernel's dependency wait for the first pages of a CTA's first unit.  L2 is the point of
// coherence, so a prefetched line can never hide a later write of the predecessor kernel.
__device__ __forceinline__ void tma_prefetch_5d(const void* tmap, int c0, int c1, int c2, int c3, int c4) {
    asm volatile("cp.async.bulk.prefetch.tensor.5d.L2.global.tile [%0, {%1, %2, %3, %4, %5}];" ::"l"(tmap), "r"(c0),
                 "r"(c1), "r"(c2), "r"(c3), "r"(c4)
                 : "memory");
}
__device__ __forceinline__ void prefetch_l2(const void* ptr) {
    asm volatile("prefetch.global.L2 [%0];" ::"l"(ptr));
}
__device__ __forceinline__ void tma_load_4d(uint32_t dst, const void* tmap, uint32_t bar, int c0, int c1,
                                            int c2, int c3) {
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes "
        "[%0], [%1, {%3, %4, %5, %6}], [%2];" ::"r"(dst),
        "l"(tmap), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
        : "memory");
}
__device__ __forceinline__ void tma_prefetch_desc(const void* tmap) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(tmap) : "memory");
}

__device__ __forceinline__ void ldmatrix_x4(uint32_t addr, uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0, %1, %2, %3}, [%4];"
                 : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3)
                 : "r"(addr)
                 : "memory");
}
__device__ __forceinline__ void ldmatrix_x4_trans(uint32_t addr, uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0, %1, %2, %3}, [%4];"
                 : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3)
                 : "r"(addr)
                 : "memory");
}
__device__ __forceinline__ uint32_t movmatrix_trans(uint32_t a) {
    uint32_t d;
    asm volatile("movmatrix.sync.aligned.m8n8.trans.b16 %0, %1;" : "=r"(d) : "r"(a));
    return d;
}
// D(16x8, f32) += A(16x16, f16, row) * B(16x8, f16, col)
__device__ __forceinline__ void mma_16816(float (&c)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3,
                                          uint32_t b0, uint32_t b1) {
    asm volatile(
        "mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, {%8, %9}, "
        "{%0, %1, %2, %3};"
        : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
        : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
// two E4M3 bytes (low 16 bits of x) -> half2, exact
__device__ __forceinline__ uint32_t cvt_e4m3x2_to_half2(uint32_t x) {
    uint32_t d;
    asm("{\n\t.reg .b16 t;\n\tcvt.u16.u32 t, %1;\n\tcvt.rn.f16x2.e4m3x2 %0, t;\n\t}" : "=r"(d) : "r"(x));
    return d;
}
// two cache bytes (low 16 bits of x) -> half2, exact.  INT8: (b ^ 0x80) | 0x6400 is the FP16 number
// 1024 + (b + 128); subtracting 1152 leaves b (integers below 2048 are exact in FP16).
template <int KVT>
__device__ __forceinline__ uint32_t cvt_bytes2_to_half2(uint32_t x) {
    if constexpr (KVT == 2) {
        const uint32_t biased = __byte_perm(x ^ 0x8080u, 0x64646464u, 0x4140);
        const __half2 h = __hsub2(*reinterpret_cast<const __half2*>(&biased), __floats2half2_rn(1152.f, 1152.f));
        return *reinterpret_cast<const uint32_t*>(&h);
    } else {
        return cvt_e4m3x2_to_half2(x);
    }
}
// two FP32 values -> two cache bytes (lo in bits 7..0, hi in bits 15..8), ONE rounding each (DESIGN.md
// reading A30).  E4M3: round to nearest even, magnitudes beyond 448 saturate (satfinite); INT8: round
// half to even, clamped to [-127, 127].
template <int KVT>
__device__ __forceinline__ uint32_t cvt_float2_to_bytes2(float lo, float hi) {
    if constexpr (KVT == 2) {
        const int a = max(-127, min(127, __float2int_rn(lo))), b = max(-127, min(127, __float2int_rn(hi)));
        return (uint32_t)(a & 0xff) | ((uint32_t)(b & 0xff) << 8);
    } else {
        unsigned short r;
        asm("cvt.rn.satfinite.e4m3x2.f32 %0, %1, %2;" : "=h"(r) : "f"(hi), "f"(lo));
        return r;
    }
}
__device__ __forceinline__ void sts_b16(uint32_t addr, uint32_t v) {
    asm volatile("st.shared.b16 [%0], %1;" ::"r"(addr), "h"((unsigned short)v) : "memory");
}
__device__ __forceinline__ uint32_t pack_half2(float lo, float hi) {
    __half2 h = __floats2half2_rn(lo, hi);
    return *reinterpret_cast<uint32_t*>(&h);
}

// ------------------------------------------------------------------ split-bound policy on the device
// (PAPER.md:63-75).  Shared by the builder kernel (pkv_aux.cu) and by the decode kernel's fused
// build (pkv_decode_tma.cu): same integer formulas as the host planner (pkv_common.h row_splits).

// A row's length as the planner uses it: negative counts as empty; with PKV_FLAG_VALIDATE a length
// the block table cannot describe is clamped to max_tokens (and reported, plan_len_fault).
__device__ __forceinline__ int32_t plan_len(const PlanArgs& a, int32_t N) {
    N = max(N, 0);
    if ((a.flags & PKV_FLAG_VALIDATE) && N > a.max_tokens) N = a.max_tokens;
    return N;
}
__device__ __forceinline__ void plan_len_fault(const PlanArgs& a, int32_t N, int32_t* error_word) {
    if (error_word && (a.flags & PKV_FLAG_VALIDATE) && N > a.max_tokens) atomicOr(error_word, (int32_t)PKV_DEVERR_SEQ_LEN);
}
// A block-table entry as the kernels use it: with PKV_FLAG_VALIDATE an id outside [0, num_pages)
// is reported and replaced by page 0 (the pool is never read out of bounds).
__device__ __forceinline__ int32_t checked_page(int32_t page, int32_t flags, int64_t num_pages, int32_t* error_word) {
    if ((flags & PKV_FLAG_VALIDATE) && (page < 0 || (int64_t)page >= num_pages)) {
        atomicOr(error_word, (int32_t)PKV_DEVERR_PAGE_ID);
        return 0;
    }
    return page;
}

struct PlanScratch {   // shared memory of the calling CTA
    int32_t warp_sums[32];
    int32_t carry, max_n, sum_n;
    unsigned long long sum_seq;
};
struct PlanTotals {
    int32_t row_slots, max_n, sum_n;   // sum_n = sum_i n_i (non-empty splits)
    long long sum_seq;
};

// BALANCED (include/pkv.h): the batch-wide chunk, computed by one warp (every lane returns it).
// lens[i] is row i's length (global or shared memory; values <= 0 count as empty rows).
// Same result as the host's balanced_chunk (pkv_common.h): `fits` is monotone in c, so the
// smallest fitting c of [lo, hi] is found either by the host's bisection (large batches: lanes
// over rows) or by testing 32 candidates at once (small batches: lanes over candidates, no
// shuffles on the critical path of a short decode step).  32-bit arithmetic while W < 2^31.
__device__ __forceinline__ int32_t balanced_chunk_warp(const PlanArgs& a, const int32_t* lens, int lane) {
    long long W64 = 0;
    for (int i = lane; i < a.B; i += 32) {
        const int N = plan_len(a, lens[i]);
        if (N > 0) W64 += (unsigned)(N + a.tile_tokens - 1) / (unsigned)a.tile_tokens;
    }
    if (__any_sync(0xffffffffu, W64 >= (1 << 26))) {   // 32 lanes x 2^26 < 2^31: else one redux.sync
#pragma unroll
        for (int off = 16; off >= 1; off >>= 1) W64 += __shfl_xor_sync(0xffffffffu, W64, off);
    } else {
        W64 = (long long)__reduce_add_sync(0xffffffffu, (unsigned)W64);
    }
    auto units_of = [&](unsigned c, int first, int step) {   // sum over rows first, first+step, ... of ceil(T_i / c)
        // ceil(T_i / c) = ceil(N_i / (tile_tokens * c)); 32-bit unsigned division
        const unsigned long long span64 = (unsigned long long)(unsigned)a.tile_tokens * c;
        const unsigned span = span64 >= 0x7fffffffull ? 0x7fffffffu : (unsigned)span64;
        unsigned units = 0;
        for (int i = first; i < a.B; i += step) {
            const int N = plan_len(a, lens[i]);
            if (N > 0) units += ((unsigned)N + span - 1u) / span;
        }
        return units;
    };
    if (W64 <= 0 || a.num_sms <= 0) return 1;
    if (W64 >= 0x7fffffffLL) {
        return balanced_chunk((int64_t)W64, a.num_sms, a.tile_tokens, [&](int32_t c) {
            unsigned units = units_of((unsigned)c, lane, 32);
#pragma unroll
            for (int off = 16; off >= 1; off >>= 1) units += __shfl_xor_sync(0xffffffffu, units, off);
            return units <= (unsigned)a.num_sms;
        });
    }
    const unsigned W = (unsigned)W64, U = (unsigned)a.num_sms;
    const unsigned m = ((unsigned)kBalMinTokens + a.tile_tokens - 1) / (unsigned)a.tile_tokens;
    const unsigned w = (W + kBalWaves * U - 1) / (kBalWaves * U);
    const unsigned c2 = w > m ? w : m;
    unsigned lo = (W + U - 1) / U, hi = lo + c2;
    if (a.B <= 16) {
        for (unsigned base = lo; base <= hi; base += 32) {
            const unsigned c = base + lane;
            const unsigned ok = __ballot_sync(0xffffffffu, c <= hi && units_of(c, 0, 1) <= U);
            if (ok) return (int32_t)(base + __ffs(ok) - 1);
        }
        return (int32_t)c2;
    }
    auto fits = [&](unsigned c) {
        unsigned units = units_of(c, lane, 32);
#pragma unroll
        for (int off = 16; off >= 1; off >>= 1) units += __shfl_xor_sync(0xffffffffu, units, off);
        return units <= U;
    };
    if (!fits(hi)) return (int32_t)c2;
    while (lo < hi) {
        const unsigned mid = (lo + hi) >> 1;
        if (fits(mid)) hi = mid; else lo = mid + 1;
    }
    return (int32_t)lo;
}

// Block-wide (every thread of the CTA calls it; blockDim.x a multiple of 32, <= 1024):
// so_out[0..B] = exclusive prefix sum of the rows' slot counts (n_i, or S on the rect route),
// len_out[i] = max(N_i, 0) if len_out != nullptr.  so_out / len_out may be global or shared.
// BALANCED: resolves the batch-wide chunk first and rewrites `a` to the FIXED_CHUNK policy it
// stands for (a.chunk_tiles = the chunk), which make_rowslot then uses.
__device__ __forceinline__ PlanTotals plan_scan(PlanArgs& a, const int32_t* seq_lens, int32_t* so_out,
                                                int32_t* len_out, PlanScratch& sc, int32_t* error_word) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nthreads = blockDim.x, nwarps = nthreads >> 5;
    const int32_t* lens = seq_lens;
    if (len_out) {   // one global round trip: stage the lengths, plan from the staged copy
        for (int i = tid; i < a.B; i += nthreads) len_out[i] = plan_len(a, __ldcg(seq_lens + request_row(a.row_index, i)));
        lens = len_out;
    }
    if (tid == 0) {
        sc.carry = 0;
        sc.max_n = 0;
        sc.sum_n = 0;
        sc.sum_seq = 0ull;
        so_out[0] = 0;
    }
    __syncthreads();
    if (a.split_mode == PKV_SPLIT_BALANCED) {
        a.chunk_tiles = balanced_chunk_warp(a, lens, lane);   // every warp computes the same value
        a.split_mode = PKV_SPLIT_FIXED_CHUNK;
    }
    for (int base = 0; base < a.B; base += nthreads) {
        const int i = base + tid;
        int32_t slots = 0, N = 0, nonempty = 0;
        if (i < a.B) {
            const int32_t raw = __ldcg(seq_lens + request_row(a.row_index, i));
            plan_len_fault(a, raw, error_word);
            N = len_out ? lens[i] : plan_len(a, raw);
            const RowSplits r = row_splits(N, a.tile_tokens, a.split_mode, a.S, a.chunk_tiles);
            nonempty = r.n;
            slots = a.route == PKV_ROUTE_WORKQUEUE ? r.n : a.S;
        }
        int32_t v = slots;   // inclusive warp scan, then scan of the warp totals
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            const int32_t u = __shfl_up_sync(0xffffffffu, v, off);
            if (lane >= off) v += u;
        }
        if (lane == 31) sc.warp_sums[warp] = v;
        __syncthreads();
        if (warp == 0) {
            int32_t w = lane < nwarps ? sc.warp_sums[lane] : 0;
#pragma unroll
            for (int off = 1; off < 32; off <<= 1) {
                const int32_t u = __shfl_up_sync(0xffffffffu, w, off);
                if (lane >= off) w += u;
            }
            sc.warp_sums[lane] = w;  // inclusive
        }
        __syncthreads();
        const int32_t incl = sc.carry + (warp > 0 ? sc.warp_sums[warp - 1] : 0) + v;
        if (i < a.B) {
            so_out[i + 1] = incl;
            atomicMax(&sc.max_n, slots);
            atomicAdd(&sc.sum_n, nonempty);
            atomicAdd(&sc.sum_seq, (unsigned long long)N);
        }
        __syncthreads();
        if (tid == nthreads - 1) sc.carry = incl;
        __syncthreads();
    }
    PlanTotals t;
    t.row_slots = sc.carry;
    t.max_n = sc.max_n;
    t.sum_n = sc.sum_n;
    t.sum_seq = (long long)sc.sum_seq;
    return t;
}

// The same plan by ONE warp (the decode kernel's planner warp; B <= a few hundred rows), in two
// parts.  plan_warp_prefix is the critical path of a decode launch: lens staged in len_out,
// BALANCED chunk resolved into `a`, so_out[0..B] by warp scans with a carry, and -- by the lane
// that owns the row -- the RowSlot of pair rs0 (the calling CTA's first work unit) into *first.
// Returns the number of (row, split) pairs.  plan_warp_totals (off the critical path) redoes the
// per-row bounds for the header counters.  so_out / len_out / first: shared memory of the CTA.
// SPEC: the lengths are read with relaxed (race-tolerant) loads before the kernel's dependency
// wait; the caller validates them after the wait (plan_lens_unchanged) and re-plans on a mismatch.
__device__ __forceinline__ int32_t ld_relaxed_s32(const int32_t* ptr) {
    int32_t v;
    asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(ptr) : "memory");
    return v;
}
template <bool SPEC = false>
__device__ __forceinline__ int32_t plan_warp_prefix(PlanArgs& a, const int32_t* seq_lens, int32_t* so_out,
                                                    int32_t* len_out, int lane, int rs0, RowSlot* first,
                                                    int32_t* error_word = nullptr) {
#pragma unroll 4
    for (int i = lane; i < a.B; i += 32) {
        const int32_t gi = !a.row_index ? i : (SPEC ? ld_relaxed_s32(a.row_index + i) : __ldcg(a.row_index + i));
        const int32_t N = SPEC ? ld_relaxed_s32(seq_lens + gi) : __ldcg(seq_lens + gi);
        if (!SPEC) plan_len_fault(a, N, error_word);
        len_out[i] = plan_len(a, N);
    }
    if (lane == 0) so_out[0] = 0;
    __syncwarp();
    if (a.split_mode == PKV_SPLIT_BALANCED) {
        a.chunk_tiles = balanced_chunk_warp(a, len_out, lane);
        a.split_mode = PKV_SPLIT_FIXED_CHUNK;
    }
    int32_t carry = 0;
    for (int base = 0; base < a.B; base += 32) {
        const int i = base + lane;
        int32_t slots = 0, N = 0;
        RowSplits r = {0, 0, 0};
        if (i < a.B) {
            N = len_out[i];
            r = row_splits(N, a.tile_tokens, a.split_mode, a.S, a.chunk_tiles);
            slots = a.route == PKV_ROUTE_WORKQUEUE ? r.n : a.S;
        }
        int32_t v = slots;
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            const int32_t u = __shfl_up_sync(0xffffffffu, v, off);
            if (lane >= off) v += u;
        }
        const int32_t incl = carry + v, excl = incl - slots;
        if (i < a.B) {
            so_out[i + 1] = incl;
            if (rs0 >= excl && rs0 < incl) {   // this lane's row owns pair rs0
                RowSlot d;
                d.row = i; d.so = excl; d.n = slots; d.split = rs0 - excl;
                int32_t tb = 0, te = 0;
                if (r.T > 0) {
                    const long long b = (long long)d.split * r.c, e = b + r.c;
                    tb = (int32_t)(b < r.T ? b : r.T);
                    te = (int32_t)(e < r.T ? e : r.T);
                }
                d.tok0 = tb * a.tile_tokens;
                d.tok1 = min(te * a.tile_tokens, N);
                d.grow = !a.row_index ? i : (SPEC ? ld_relaxed_s32(a.row_index + i) : __ldcg(a.row_index + i));
                d.nlen = N;
                *first = d;
            }
        }
        carry += __shfl_sync(0xffffffffu, v, 31);
    }
    __syncwarp();
    return carry;
}

// After the dependency wait: are the lengths a speculative plan was made from (len_s) still the
// ones in memory?  Every lane returns the answer.
__device__ __forceinline__ bool plan_lens_unchanged(const PlanArgs& a, const int32_t* seq_lens, const int32_t* len_s,
                                                    int lane, int32_t* error_word = nullptr) {
    bool same = true;
    for (int i = lane; i < a.B; i += 32) {
        const int32_t N = __ldcg(seq_lens + request_row(a.row_index, i));
        plan_len_fault(a, N, error_word);
        same &= plan_len(a, N) == len_s[i];
    }
    return __all_sync(0xffffffffu, same);
}

__device__ __forceinline__ PlanTotals plan_warp_totals(const PlanArgs& a, const int32_t* len_s, int32_t row_slots,
                                                       int lane) {
    int32_t max_n = 0, sum_n = 0;
    long long sum_seq = 0;
    for (int i = lane; i < a.B; i += 32) {
        const int32_t N = len_s[i];
        const RowSplits r = row_splits(N, a.tile_tokens, a.split_mode, a.S, a.chunk_tiles);
        sum_n += r.n;
        sum_seq += N;
        max_n = max(max_n, a.route == PKV_ROUTE_WORKQUEUE ? r.n : a.S);
    }
#pragma unroll
    for (int off = 16; off >= 1; off >>= 1) {
        max_n = max(max_n, __shfl_xor_sync(0xffffffffu, max_n, off));
        sum_n += __shfl_xor_sync(0xffffffffu, sum_n, off);
        sum_seq += __shfl_xor_sync(0xffffffffu, sum_seq, off);
    }
    PlanTotals t;
    t.row_slots = row_slots;
    t.max_n = max_n;
    t.sum_n = sum_n;
    t.sum_seq = sum_seq;
    return t;
}

// The (row, split) pair rs: the row by binary search in so[0..B], bounds from the row's length.
// `lens` is indexed by row (seq_lens itself, or the clamped copy plan_scan made).
__device__ __forceinline__ RowSlot make_rowslot(const PlanArgs& a, const int32_t* so, const int32_t* lens, int rs,
                                                int32_t* t_begin, int32_t* t_end) {
    int lo = 0, hi = a.B - 1;
    while (lo < hi) {   // largest row with so[row] <= rs
        const int mid = (lo + hi + 1) >> 1;
        if (so[mid] <= rs) lo = mid; else hi = mid - 1;
    }
    RowSlot d;
    d.row = lo;
    d.so = so[lo];
    d.n = so[lo + 1] - d.so;
    d.split = rs - d.so;
    const int32_t N = plan_len(a, lens[lo]);
    const RowSplits r = row_splits(N, a.tile_tokens, a.split_mode, a.S, a.chunk_tiles);
    int32_t tb = 0, te = 0;
    if (r.T > 0) {
        const long long b = (long long)d.split * r.c, e = (long long)(d.split + 1) * r.c;
        tb = (int32_t)(b < r.T ? b : r.T);
        te = (int32_t)(e < r.T ? e : r.T);
    }
    d.tok0 = tb * a.tile_tokens;
    d.tok1 = min(te * a.tile_tokens, N);
    d.grow = request_row(a.row_index, lo);
    d.nlen = N;
    *t_begin = tb;
    *t_end = te;
    return d;
}

// Writes pair rs's RowSlot and its Hkv task entries (canonical order: so*Hkv + g*n + s).
__device__ __forceinline__ void write_pair(const PlanArgs& a, const RowSlot& d, int32_t tb, int32_t te, int rs,
                                          RowSlot* rowslots, pkv_task* tasks, int64_t tasks_cap) {
    rowslots[rs] = d;
    for (int g = 0; g < a.Hkv; ++g) {
        const int64_t idx = (int64_t)d.so * a.Hkv + (int64_t)g * d.n + d.split;
        if (idx < tasks_cap) {
            pkv_task t;
            t.row = d.row; t.kvh = g; t.split = d.split; t.t_begin = tb; t.t_end = te;
            tasks[idx] = t;
        }
    }
}

// ------------------------------------------------------------------ merge of split states

// Exact merge of the n states of one (row, kvh, head-in-group hh), stored at
// slots slot_base .. slot_base+n-1, by ONE warp -- the fused in-kernel merge of PAPER.md:77 (the
// separate merge kernel, pkv_aux.cu, spreads a row over a whole CTA instead):
//   M   = max_s m_s
//   P_k = sum over s = k, k+4, k+8, ... (ascending) of exp(m_s - M) * (l_s, a_s),   k = 0..3
//   (L, A) = ((P_0 + P_1) + P_2) + P_3,   O = A / L,   LSE = M + log L
// Lane owns channels 4*lane .. 4*lane+3 (one 16-byte load per state row).  Neutral states
// (m = -inf, l = 0) drop out; all-neutral gives O = 0, LSE = -inf.

template <int G>
__device__ __forceinline__ float merge_row_max(const DecodeParams& p, int64_t slot_base, int n, int hh, int lane) {
    float M = -INFINITY;
    for (int s = lane; s < n; s += 32) M = fmaxf(M, __ldcg(p.part_m + (slot_base + s) * G + hh));
#pragma unroll
    for (int off = 16; off >= 1; off >>= 1) M = fmaxf(M, __shfl_xor_sync(0xffffffffu, M, off));
    return M;
}

// NK interleaved partial sums of one lane's 4 channels over the states first, first+stride, ...
// kMergeBatch independent state loads are in flight per lane; they bypass L1 (states are written
// by other SMs, in the fused path during this very launch).
constexpr int kMergeBatch = 8;
template <int G, int NK>
__device__ __forceinline__ void merge_accumulate(const DecodeParams& p, int64_t slot_base, int n, int hh, float M,
                                                 int first, int stride, int ch, float (&L)[NK], float4 (&A)[NK]) {
#pragma unroll
    for (int k = 0; k < NK; ++k) {
        L[k] = 0.f;
        A[k] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    const int cnt = n > first ? (n - first + stride - 1) / stride : 0;
    for (int i0 = 0; i0 < cnt; i0 += kMergeBatch) {
        float mv[kMergeBatch], lv[kMergeBatch];
        float4 av[kMergeBatch];
#pragma unroll
        for (int j = 0; j < kMergeBatch; ++j) {
            const bool ok = i0 + j < cnt;
            const int64_t r = (slot_base + first + (int64_t)(ok ? i0 + j : 0) * stride) * G + hh;
            mv[j] = ok ? __ldcg(p.part_m + r) : -INFINITY;
            lv[j] = ok ? __ldcg(p.part_l + r) : 0.f;
            av[j] = ok ? __ldcg(reinterpret_cast<const float4*>(p.part_acc + r * p.d + ch))
                       : make_float4(0.f, 0.f, 0.f, 0.f);
        }
#pragma unroll
        for (int j = 0; j < kMergeBatch; ++j) {
            const float w = ex2_approx((mv[j] - M) * kLog2e);  // exp2(-inf) = 0
            const int k = NK == 4 ? (j & 3) : 0;
            L[k] = fmaf(w, lv[j], L[k]);
            A[k].x = fmaf(w, av[j].x, A[k].x); A[k].y = fmaf(w, av[j].y, A[k].y);
            A[k].z = fmaf(w, av[j].z, A[k].z); A[k].w = fmaf(w, av[j].w, A[k].w);
        }
    }
}

// Stores four channels ch .. ch+3 of output row o (FP16) and, by the lane with store_lse, its LSE.
__device__ __forceinline__ void merge_store(const DecodeParams& p, int64_t o, int ch, bool store_lse, float M, float L,
                                            float4 A) {
    __half2* dst = reinterpret_cast<__half2*>(p.out + o * p.d + ch);
    if (M == -INFINITY) {  // no state or only neutral states (A9)
        dst[0] = __floats2half2_rn(0.f, 0.f);
        dst[1] = __floats2half2_rn(0.f, 0.f);
        if (p.lse && store_lse) p.lse[o] = -INFINITY;
        return;
    }
    const float inv = 1.0f / L;
    dst[0] = __floats2half2_rn(A.x * inv, A.y * inv);
    dst[1] = __floats2half2_rn(A.z * inv, A.w * inv);
    if (p.lse && store_lse) p.lse[o] = M + logf(L);
}

// One warp merges head hh completely (fused path; also any caller without helpers).
template <int G>
__device__ __forceinline__ void merge_head_warp(const DecodeParams& p, int64_t slot_base, int n, int orow, int kvh,
                                                int hh, int lane) {
    const float M = merge_row_max<G>(p, slot_base, n, hh, lane);
    // slabs of 128 channels: one for d = 64 (half the lanes) and 128, two for d = 256
    for (int ch = lane * 4; ch < p.d; ch += 128) {
        float L[4];
        float4 A[4];
        merge_accumulate<G, 4>(p, slot_base, n, hh, M, 0, 1, ch, L, A);
        const float Ls = ((L[0] + L[1]) + L[2]) + L[3];
        float4 As;
        As.x = ((A[0].x + A[1].x) + A[2].x) + A[3].x;
        As.y = ((A[0].y + A[1].y) + A[2].y) + A[3].y;
        As.z = ((A[0].z + A[1].z) + A[2].z) + A[3].z;
        As.w = ((A[0].w + A[1].w) + A[2].w) + A[3].w;
        merge_store(p, (int64_t)orow * p.Hq + kvh * G + hh, ch, ch == 0, M, Ls, As);
    }
}

// ------------------------------------------------------------------ task epilogue

// Shared-memory combine buffer of one CTA: every compute warp leaves the state of its share of
// a task's tokens in its own row; m in raw-dot units (x = scale * raw).
// acc rows hold D + 4 floats: (D + 4) % 32 = 4 spreads the banks
template <int G, int NWTOT, int D = kD>
struct CombineBuf {
    float acc[NWTOT][G][D + 4];
    float m[NWTOT][G < 8 ? 8 : G];
    float l[NWTOT][G < 8 ? 8 : G];
    int flag[NWTOT];
};

template <int NW>
__device__ __forceinline__ void group_sync(int bar_id) {
    if (NW == 1) __syncwarp(); else named_bar_sync(bar_id, NW * 32);
}

// FUSED merge tail: a group of NW warps has stored split `split` of (row, kvh); the
// group that completes the last of the n_i splits (atomic completion counter, self-resetting for
// graph replay) merges the row's slot range in place.  flag = a shared-memory word of the group.
// `arrivals`: groups that complete one split of (row, kvh) between them (2 when G = 16: one group
// per block of 8 query heads); the last of the n_i * arrivals merges all G heads.
template <int G, int NW>
__device__ __forceinline__ void fused_complete(const DecodeParams& p, int* flag, int row, int orow, int kvh, int split,
                                               int n_i, int64_t slot, int gtid, int bar_id, int arrivals = 1) {
    __threadfence();  // partial state visible device-wide before the completion count
    group_sync<NW>(bar_id);
    if (gtid == 0) {
        const int old = atomicAdd(&p.fuse_counters[row * p.Hkv + kvh], 1);
        const int last = (old == n_i * arrivals - 1);
        if (last) p.fuse_counters[row * p.Hkv + kvh] = 0;
        *flag = last;
    }
    group_sync<NW>(bar_id);
    if (*flag) {
        __threadfence();
        const int64_t base = slot - split;  // first slot of (row, kvh): DESIGN.md A8
        for (int hh = gtid >> 5; hh < G; hh += NW) merge_head_warp<G>(p, base, n_i, orow, kvh, hh, gtid & 31);
    }
    group_sync<NW>(bar_id);  // flag may be rewritten after this
}

// Writes an empty task's result (rect route): neutral partial state, or zeros when
// the row has a single slot (direct output).  Called by the NW warps that own the task.
// The group owns query heads h0 .. h0+GW-1 of the KV head's G (GW = G, h0 = 0 unless G = 16).
template <int G, int NW, int GW = G>
__device__ __forceinline__ void store_empty_task(const DecodeParams& p, int* flag, int row, int orow, int kvh, int split,
                                                 int n_i, int64_t slot, int gtid, int bar_id, int h0 = 0) {
    const int dsh = __ffs(p.d) - 1;   // d is a power of two
    for (int idx = gtid; idx < (GW << dsh); idx += NW * 32) {
        const int hh = h0 + (idx >> dsh), dd = idx & (p.d - 1);
        if (n_i <= 1) {
            const int64_t o = (int64_t)orow * p.Hq + kvh * G + hh;
            p.out[o * p.d + dd] = __float2half_rn(0.f);
            if (p.lse && dd == 0) p.lse[o] = -INFINITY;
        } else {
            p.part_acc[(slot * G + hh) * p.d + dd] = 0.f;
            if (dd == 0) {
                p.part_m[slot * G + hh] = -INFINITY;
                p.part_l[slot * G + hh] = 0.f;
            }
        }
    }
    if (n_i > 1 && p.merge_mode == PKV_MERGE_FUSED)
        fused_complete<G, NW>(p, flag, row, orow, kvh, split, n_i, slot, gtid, bar_id, G / GW);
}

// A group of NW warps (rows w0, w0+wstride, ... of `cb`) has processed one task.  Combines the
// NW warp states and stores the task's result: direct FP16 output when the row has one split,
// else the FP32 partial state in its compact slot; in FUSED mode
// the group that completes the last split of (row, kvh) merges in place.
// gtid = 0..NW*32-1 within the group; the group synchronises with group_sync<NW>(bar_id); the
// caller has synchronised after filling `cb`.
template <int G, int NW, int NWTOT, int GW = G, int D = kD>
__device__ __forceinline__ void finalize_task(const DecodeParams& p, CombineBuf<GW, NWTOT, D>& cb, int w0, int wstride,
                                              int row, int orow, int kvh, int split, int n_i, int64_t slot, int gtid,
                                              int bar_id, int h0, float sc, float sc2) {
    // sc = scale of the raw dot products in cb.m (x = sc * raw), sc2 = sc * log2(e)
    for (int idx = gtid; idx < GW * D; idx += NW * 32) {
        const int hh = idx / D, dd = idx % D;   // head within the group's block; h0 + hh within the KV head
        float M = -INFINITY;
#pragma unroll
        for (int i = 0; i < NW; ++i) M = fmaxf(M, cb.m[w0 + i * wstride][hh]);
        float L = 0.f, A = 0.f;
#pragma unroll
        for (int i = 0; i < NW; ++i) {
            const int w = w0 + i * wstride;
            const float wgt = ex2_approx((cb.m[w][hh] - M) * sc2);  // m = -inf -> 0
            L += wgt * cb.l[w][hh];
            A += wgt * cb.acc[w][hh][dd];
        }
        if (n_i <= 1) {
            const int64_t o = (int64_t)orow * p.Hq + kvh * G + h0 + hh;
            p.out[o * D + dd] = __float2half_rn(A / L);
            if (p.lse && dd == 0) p.lse[o] = M * sc + logf(L);
        } else {
            p.part_acc[(slot * G + h0 + hh) * D + dd] = A;
            if (dd == 0) {
                p.part_m[slot * G + h0 + hh] = M * sc;
                p.part_l[slot * G + h0 + hh] = L;
            }
        }
    }
    if (n_i > 1 && p.merge_mode == PKV_MERGE_FUSED)
        fused_complete<G, NW>(p, &cb.flag[w0], row, orow, kvh, split, n_i, slot, gtid, bar_id, G / GW);
    group_sync<NW>(bar_id);  // cb rows may be refilled after this
}

// Rows with N_i = 0 emit no task in the workqueue route: out = 0, lse = -inf (A9).
__device__ __forceinline__ void zero_empty_rows(const DecodeParams& p) {
    const int per_row = p.Hq * p.d;
    for (int i = blockIdx.x; i < p.B; i += gridDim.x) {
        const int64_t gi = request_row(p.row_index, i);
        if (p.seq_lens[gi] > 0) continue;
        for (int e = threadIdx.x; e < per_row; e += blockDim.x) {
            p.out[gi * per_row + e] = __float2half_rn(0.f);
            if (p.lse && e < p.Hq) p.lse[gi * p.Hq + e] = -INFINITY;
        }
    }
}

// Launch with the programmatic-stream-serialization attribute: in a stream (and in a captured
// graph) the kernel may start while its predecessor is still running; it orders itself with
// pdl_wait().  pdl = false (PKV_FLAG_NO_PDL) is a plain launch.
template <typename... KArgs, typename... Args>
cudaError_t launch_pdl(bool pdl, void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream,
                       Args&&... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kernel, std::forward<Args>(args)...);
}

inline PlanArgs make_plan_args(const pkv_shape& shape, const Resolved& rp) {
    PlanArgs a;
    a.B = shape.B; a.Hkv = shape.Hkv; a.S = rp.S; a.tile_tokens = rp.tile_tokens;
    a.split_mode = rp.split_mode; a.chunk_tiles = rp.chunk_tiles; a.route = rp.route; a.num_sms = rp.num_sms;
    a.flags = rp.flags;
    const int64_t mt = (int64_t)shape.max_pages * shape.page_size;
    a.max_tokens = (int32_t)(mt < 0x7fffffff ? mt : 0x7fffffff);
    a.row_index = nullptr;
    return a;
}

// launchers implemented in the .cu files
cudaError_t launch_decode_simt(const DecodeParams& p, int G, int grid, cudaStream_t stream);
cudaError_t launch_decode_tma(const DecodeParams& p, int G, int HG, int D, int kvt, int grid, const void* tmap_k,
                              const void* tmap_v, cudaStream_t stream);
cudaError_t launch_builder(const pkv_shape& shape, const Resolved& rp, const int32_t* seq_lens_dev,
                           const int32_t* row_index, QueueHeader* hdr, int32_t* split_offsets, int32_t* fuse_counters, RowSlot* rowslots,
                           pkv_task* tasks, int64_t tasks_cap, cudaStream_t stream);
cudaError_t launch_merge(const DecodeParams& p, int G, cudaStream_t stream);
// pkv_decode_host_pipelined (pkv_aux.cu): the gate / stage kernel and the completion signal.
constexpr int kMaxStageSegs = 4;
constexpr int kStageThreads = 1024;           // 16 KiB of inputs in one round of 16-byte loads over the host link
constexpr size_t kMaxStageBytes = 256 << 10;  // beyond this the copy engine is the faster way up
struct StageSegs {
    uint32_t off[kMaxStageSegs];      // byte offset in the image, multiple of 16
    uint32_t chunks[kMaxStageSegs];   // 16-byte chunks
    int32_t n;
};
// 32-bit words of the pipeline in the pinned, device-mapped image header (pkv_api.cu PipeWords)
constexpr int kPipeFlagWord = 0;      // host -> GPU: number of the last released step
constexpr int kPipeStagedWord = 16;   // GPU -> host: the stage kernel of step n has read the image
constexpr int kPipeDoneWord = 17;     //              step n's result is in out_host
constexpr int kPipeExpiredWord = 18;  //              step n was never released: it ran on stale inputs
cudaError_t launch_stage(const void* src_mapped, void* dst, const StageSegs& segs, uint32_t* words_mapped, uint32_t seq, bool gate,
                         unsigned long long timeout_ns, cudaStream_t stream);
constexpr int kSignalThreads = 512;
cudaError_t launch_signal(uint32_t* words_mapped, uint32_t seq, bool pdl, const void* out_dev, void* out_host_mapped, size_t out_bytes,
                          cudaStream_t stream);
int decode_tma_stage_bytes(int HG, int D, bool fp8);

}  // namespace pkv
