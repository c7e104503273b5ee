// pkv_decode_tma.cu -- PKV_KERNEL_TMA_MMA: the B200 decode kernel.
//
// Persistent, warp-specialised CTA, one per SM.  The paper maps one CTA to one (request, KV head,
// split) work item; here a resident CTA walks many work UNITS, a unit being the HG
// tasks (row, kvh = hg*HG .. hg*HG+HG-1, split) of the workqueue that share a tile interval
// (DESIGN.md "CTA mapping").  With HG = Hkv = 8 a unit streams whole pages: one page of K (or V)
// is ONE contiguous 32 KiB TMA box in the default [page, token, head, d] layout.
//
//   producer warps (NP)  producer 0 takes units (first by block index, then from an atomic
//                        counter when every head has one compute warp, else round-robin: see
//                        pkv_api.cu), resolves (row, split) and publishes the unit on a small
//                        ring.  Every producer walks its share of the unit's slice of the
//                        block table (PAPER.md:50 page accessor), 32 entries per load, and per
//                        page issues one TMA box for K and one for V -- 16 tokens x HG heads x
//                        128 channels, 128-byte swizzled -- into a ring of stages guarded by
//                        full(K)/full(V)/empty mbarriers.  Producers run ahead across unit
//                        boundaries, so the ring never drains between units.
//   compute warps (8)    warp cw serves head cw % HG; the 8/HG warps of a head take pages
//                        round-robin.  Per page and head:
//                          S^T[16 tok x 8 heads] = K[16 x 128] . Q^T      8 HMMA m16n8k16
//                          exact online softmax in FP32, P -> FP16
//                          O^T[128 x 8 heads]  += V^T[128 x 16] . P^T     8 HMMA m16n8k16
//                        Tokens sit on the MMA M axis and the G <= 8 grouped query heads
//                         on the N = 8 axis, so G = 8 fills the tile and G = 4
//                        half of it; K is read with ldmatrix, V with ldmatrix.trans, P^T is
//                        made from the S^T accumulator layout with movmatrix.
//   unit end             with one warp per head the state goes from the MMA accumulators straight
//                        to the task's partial-state slot (or, for a row with a single split, to
//                        `out`); several warps per head combine through shared memory first
//                        (pkv_device.cuh finalize_task).
//   fused build          producer 0 derives the plan from seq_lens inside the kernel (split-bound
//                        policy: one load round trip + warp scans) together with
//                        this CTA's first unit; the planner warp (1) takes the plan from shared
//                        memory and writes the CTA's share of the bit-exact queue off everybody's
//                        critical path.
// K/V loads carry an L2 evict_first policy: the stream is read once per step, the step's small
// re-read data (seq_lens, block table, q, partial states) stays in L2.
#include <cuda.h>

#include "pkv_device.cuh"

namespace pkv {

namespace {

constexpr int kComputeWarps = 8;
constexpr int kPlanBar = 9;         // named barrier: planner warp -> producer 0 (1..8 belong to the head groups)
constexpr int kPatchBar0 = 10;      // named barriers 10..13: fused append with G = 16, the two warps that share a stage
constexpr int kRing = 4;            // unit ring between producer 0 and everybody else
constexpr int kMaxStages = 24;

__host__ __device__ constexpr int producers_for(int HG) { return HG >= 4 ? 1 : (HG == 2 ? 2 : 4); }

struct UnitInfo {
    int unit;   // -1: no more work
    int row, so, n, split, tok0, tok1;   // the unit's RowSlot
    int grow;   // request row: the row of q, out, lse and block_table (= row unless the launch is indexed)
    int nlen;   // the row's length N_i
};

template <int G, int D>
struct SmemTail {
    CombineBuf<G, kComputeWarps, D> cb;
    unsigned long long full_k[kMaxStages];
    unsigned long long full_v[kMaxStages];
    unsigned long long empty_bar[kMaxStages];
    unsigned long long ring_full[kRing];
    unsigned long long ring_empty[kRing];
    UnitInfo ring[kRing];
    int32_t plan_row_slots;            // fused build: totals handed from the planner warp to producer 0
    int32_t plan_chunk;
    RowSlot first_slot;                // the RowSlot of this CTA's first unit (planner -> producer 0)
    uint32_t sink_f[kComputeWarps];    // dependency sinks (see "stage release" in the kernel)
    int sink_i[16];
    int32_t so_s[kMaxFusedRows + 1];   // fused build: split_offsets
    int32_t len_s[kMaxFusedRows];      //              max(N_i, 0)
};

// G = 16 is two blocks of 8 query heads (the MMA's N = 8 columns): NBK column blocks of GW heads,
// each with warps of its own that share the streamed K/V stage.
__host__ __device__ constexpr int blocks_for(int G) { return G > 8 ? G / 8 : 1; }

// One stage = one block of 16 tokens of HG heads: K (16 x D halves) then V, per head D * 32 bytes each.
// FP8 caches: one byte per channel, half the bytes.
__host__ __device__ constexpr int stage_bytes_for(int HG, int D, bool fp8 = false) { return HG * D * (fp8 ? 32 : 64); }

template <int G, int HG, int D, bool FP8 = false>   // FP8: one-byte caches (E4M3 or INT8)
__host__ __device__ constexpr int stages_for() {
    // 227 KiB per CTA, minus the tail, minus 1 KiB alignment slack
    constexpr int avail = 232448 - 1024 - (int)sizeof(SmemTail<G / blocks_for(G), D>);
    constexpr int n = avail / stage_bytes_for(HG, D, FP8);
    // Stage s always belongs to producer s % NP and, per head, to compute warp s % WPH (see the
    // kernel): any stage count works, the shares differ by at most one stage.
    return n > kMaxStages ? kMaxStages : n;
}

// Fused KV-append (reading A29): row `orow`'s new token (position pos, row `r` = pos % 16 of
// its 16-token block) for KV head kvh.  One warp: lane pairs channels (c, c+1) with (c + D/2, c + D/2 + 1),
// rotates K in FP32 (product by product, as the oracle), and stores the FP16 result both into the
// head's block of the shared-memory stage `sb` (128-byte swizzled rows of 64 channels) and into the
// pool at the token's slot.  V is copied unrotated.
template <int D, bool IS_K>
__device__ __forceinline__ void append_patch(const DecodeParams& p, uint32_t sb, int orow, int kvh, int pos, int r, int lane,
                                             int page_shift) {
    const __half* src = (IS_K ? p.k_new : p.v_new) + ((int64_t)orow * p.Hkv + kvh) * D;
    __half* pool = const_cast<__half*>(IS_K ? p.k_cache : p.v_cache);
    const int psz = 16 << page_shift;
    const int64_t page = __ldg(p.block_table + (int64_t)orow * p.max_pages + (pos >> (4 + page_shift)));
    __half* dst = pool + page * p.stride_page + (int64_t)(pos & (psz - 1)) * p.stride_token + (int64_t)kvh * p.stride_head;
    const bool rot = IS_K && p.rope_cos != nullptr && pos < p.rope_positions;
    for (int c = lane * 2; c < D / 2; c += 64) {
        __half2 lo = *reinterpret_cast<const __half2*>(src + c);
        __half2 hi = *reinterpret_cast<const __half2*>(src + c + D / 2);
        if (rot) {
            const float2 cs2 = __ldg(reinterpret_cast<const float2*>(p.rope_cos + (int64_t)pos * (D / 2) + c));
            const float2 sn2 = __ldg(reinterpret_cast<const float2*>(p.rope_sin + (int64_t)pos * (D / 2) + c));
            const float2 x1 = __half22float2(lo), x2 = __half22float2(hi);
            lo = __floats2half2_rn(__fsub_rn(__fmul_rn(x1.x, cs2.x), __fmul_rn(x2.x, sn2.x)),
                                   __fsub_rn(__fmul_rn(x1.y, cs2.y), __fmul_rn(x2.y, sn2.y)));
            hi = __floats2half2_rn(__fadd_rn(__fmul_rn(x2.x, cs2.x), __fmul_rn(x1.x, sn2.x)),
                                   __fadd_rn(__fmul_rn(x2.y, cs2.y), __fmul_rn(x1.y, sn2.y)));
        }
#pragma unroll
        for (int hf = 0; hf < 2; ++hf) {
            const int ch = c + hf * (D / 2);
            const __half2 val = hf ? hi : lo;
            // stage: 64-channel block ch / 64, row r, 16-byte chunk ((ch % 64) / 8) ^ (r % 8), byte (ch % 8) * 2
            const uint32_t a = sb + (ch >> 6) * 2048 + r * 128 + (((((ch & 63) >> 3) ^ (r & 7))) << 4) + (ch & 7) * 2;
            sts_b32(a, *reinterpret_cast<const uint32_t*>(&val));
            *reinterpret_cast<__half2*>(dst + ch) = val;
        }
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // the stage is refilled by the async proxy later
    __syncwarp();
}

// The same for one-byte caches (d = 128; reading A30): the token is rotated as above (FP16
// result), divided by its head's scale in FP32 and rounded once to the cache's code; the code bytes go
// into the head's block of the stage (one 128-byte swizzled row of 128 channels per token) and into
// the pool.  A lane owns channels (c, c+1) and (c + 64, c + 65), c = 2 * lane.
template <int KVT, bool IS_K>
__device__ __forceinline__ void append_patch_q8(const DecodeParams& p, uint32_t sb, int orow, int kvh, int pos, int r, int lane,
                                                int page_shift) {
    constexpr int D = 128;
    const __half* src = (IS_K ? p.k_new : p.v_new) + ((int64_t)orow * p.Hkv + kvh) * D;
    unsigned char* pool = reinterpret_cast<unsigned char*>(const_cast<__half*>(IS_K ? p.k_cache : p.v_cache));
    const float* scales = IS_K ? p.k_scale : p.v_scale;
    const float hs = scales ? __ldg(scales + kvh) : 1.f;
    const int psz = 16 << page_shift;
    const int64_t page = __ldg(p.block_table + (int64_t)orow * p.max_pages + (pos >> (4 + page_shift)));
    unsigned char* dst = pool + page * p.stride_page + (int64_t)(pos & (psz - 1)) * p.stride_token + (int64_t)kvh * p.stride_head;
    const bool rot = IS_K && p.rope_cos != nullptr && pos < p.rope_positions;
    const int c = lane * 2;
    __half2 lo = *reinterpret_cast<const __half2*>(src + c);
    __half2 hi = *reinterpret_cast<const __half2*>(src + c + D / 2);
    if (rot) {
        const float2 cs2 = __ldg(reinterpret_cast<const float2*>(p.rope_cos + (int64_t)pos * (D / 2) + c));
        const float2 sn2 = __ldg(reinterpret_cast<const float2*>(p.rope_sin + (int64_t)pos * (D / 2) + c));
        const float2 x1 = __half22float2(lo), x2 = __half22float2(hi);
        lo = __floats2half2_rn(__fsub_rn(__fmul_rn(x1.x, cs2.x), __fmul_rn(x2.x, sn2.x)),
                               __fsub_rn(__fmul_rn(x1.y, cs2.y), __fmul_rn(x2.y, sn2.y)));
        hi = __floats2half2_rn(__fadd_rn(__fmul_rn(x2.x, cs2.x), __fmul_rn(x1.x, sn2.x)),
                               __fadd_rn(__fmul_rn(x2.y, cs2.y), __fmul_rn(x1.y, sn2.y)));
    }
#pragma unroll
    for (int hf = 0; hf < 2; ++hf) {
        const int ch = c + hf * (D / 2);
        const float2 x = __half22float2(hf ? hi : lo);
        const uint32_t code = cvt_float2_to_bytes2<KVT>(__fdiv_rn(x.x, hs), __fdiv_rn(x.y, hs));
        // stage: row r, 16-byte chunk (ch / 16) ^ (r % 8), byte ch % 16
        sts_b16(sb + r * 128 + ((((ch >> 4) ^ (r & 7))) << 4) + (ch & 15), code);
        *reinterpret_cast<unsigned short*>(dst + ch) = (unsigned short)code;
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // the stage is refilled by the async proxy later
    __syncwarp();
}

// KVT: pkv_kv_dtype of the caches (0 FP16, 1 FP8 E4M3, 2 INT8); "FP8" below means any one-byte cache.
// APP: the fused KV-append (+RoPE) step (pkv_decode_append); compiled apart because its extra live
// values cost the plain step 21 registers and 0.17 us (config 2: 23.83 vs 23.66 us).
template <int G, int HG, int D, int KVT, bool APP>
__global__ void __launch_bounds__((producers_for(HG) + kComputeWarps + 1) * 32, 1)
    pkv_decode_tma_kernel(const DecodeParams p, const __grid_constant__ CUtensorMap tmap_k,
                          const __grid_constant__ CUtensorMap tmap_v) {
    constexpr bool FP8 = KVT != 0;
    static_assert(!APP || D == 128, "fused append: d = 128");
    static_assert(!FP8 || D == 128, "one-byte caches: one 128-byte swizzled row per token and head");
    constexpr int kStages = stages_for<G, HG, D, FP8>();
    constexpr int kHeadBytes = D * (FP8 ? 16 : 32);   // one head's 16 tokens x D channels of K (or V): blocks of 2 KiB
    constexpr int kStageBytes = stage_bytes_for(HG, D, FP8);   // K: HG x kHeadBytes | V: HG x kHeadBytes
    constexpr int KK = D / 16;               // k-steps of S = K.Q^T and m-tiles of O^T = V^T.P^T
    constexpr int NP = producers_for(HG);
    constexpr int NBK = blocks_for(G);       // blocks of query heads per KV head (2 when G = 16)
    constexpr int GW = G / NBK;              // query heads one warp tracks (the MMA's N columns)
    constexpr int NGRP = HG * NBK;           // (head, block) groups per CTA
    constexpr int WPH = kComputeWarps / NGRP;  // warps per group: they split the unit's pages
    constexpr int kPlanWarp = NP + kComputeWarps;   // the last warp plans and writes the queue
    static_assert(kStages >= 2, "ring too small");
    static_assert(NGRP <= kComputeWarps, "G = 16 streams at most 4 KV heads per CTA");
    extern __shared__ unsigned char smem_raw[];
    // 128-byte swizzle: every 2 KiB half-box must start on a 1024-byte boundary
    unsigned char* smem = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    SmemTail<GW, D>& tail = *reinterpret_cast<SmemTail<GW, D>*>(smem + (size_t)kStages * kStageBytes);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const uint32_t stage_base = smem_u32(smem);
    const uint32_t fullk0 = smem_u32(&tail.full_k[0]);
    const uint32_t fullv0 = smem_u32(&tail.full_v[0]);
    const uint32_t empty0 = smem_u32(&tail.empty_bar[0]);
    const uint32_t rfull0 = smem_u32(&tail.ring_full[0]);
    const uint32_t rempty0 = smem_u32(&tail.ring_empty[0]);

    if (tid == 0) PKV_TRACE_STAMP(p, 0);
    pdl_launch_dependents();
    if (tid == 0) {
        for (int s = 0; s < kStages; ++s) {
            mbar_init(fullk0 + 8 * s, 1);
            mbar_init(fullv0 + 8 * s, 1);
            mbar_init(empty0 + 8 * s, NGRP);  // one arrival per (head, block) group of the page
        }
        for (int r = 0; r < kRing; ++r) {
            mbar_init(rfull0 + 8 * r, 1);
            mbar_init(rempty0 + 8 * r, kComputeWarps + NP - 1);
        }
        mbar_fence_init();
        tma_prefetch_desc(&tmap_k);
        tma_prefetch_desc(&tmap_v);
    }
    __syncthreads();
    const int HGn = p.Hkv / HG;                               // head groups per (row, split)
    int num_units = 0;
    int early_row = -1, early_tok0 = 0, early_tok1 = 0, early_mine = 0;   // producer 0: first unit's table entries
    const int pgs = p.page_shift, pmask = (1 << pgs) - 1;   // page = 1 << ps blocks of 16 tokens
    PlanArgs plan = p.plan;   // BALANCED: the planner resolves the batch-wide chunk
    // Speculative plan.  A decode CTA is usually resident a few microseconds before its dependency
    // wait returns (programmatic launch), and the plan -- ~1 us with a fixed split count, ~2.5 us
    // BALANCED; straight-line integer code that runs once per launch -- would otherwise sit on
    // the critical path of the first TMA load.  Producer 0 makes it now from a race-tolerant read
    // of seq_lens and, after the wait, only checks that the lengths are still the same (they
    // are, unless the kernel right before this one wrote them; then it plans again).
    PlanArgs spec_plan = plan;
    int32_t spec_row_slots = 0;
    if (p.fused_build && warp == 0)
        spec_row_slots = plan_warp_prefix<true>(spec_plan, p.seq_lens, tail.so_s, tail.len_s, lane,
                                                (int)blockIdx.x / HGn, &tail.first_slot);
    if (p.force_replan && p.fused_build && warp == 0) {   // test hook: leave a wrong plan behind
        for (int i = lane; i <= p.B; i += 32) tail.so_s[i] = 0x3fffffff;
        for (int i = lane; i < p.B; i += 32) tail.len_s[i] = 1;
        if (lane == 0) tail.first_slot.tok1 = 0;
        __syncwarp();
    }
    // L2 prefetch.  Until the wait below returns the memory system is
    // underused -- the predecessor's last CTAs are draining, the merge of the previous decode step
    // is a handful of dependent round trips -- while this CTA already knows, from the speculative
    // plan, which pages it will stream first.  Producer 0 looks at those block-table entries
    // (race-tolerant loads) and asks for the pages' K/V boxes, and the unit's q rows, to be brought
    // into L2.  Nothing enters the program: L2 is the point of coherence, every value is loaded after
    // the wait; a stale guess only costs bandwidth.
    if (p.fused_build && warp == 0 && p.prefetch_pages > 0 && (int)blockIdx.x < spec_row_slots * HGn) {
        const RowSlot d = tail.first_slot;
        const int p0 = d.tok0 >> 4;   // in blocks of 16 tokens (a page holds 1 << page_shift of them)
        int np = d.tok0 < d.tok1 ? ((d.tok1 + 15) >> 4) - p0 : 0;
        np = min(min(np, p.prefetch_pages), (p.max_pages << pgs) - p0);
        if (d.row >= 0 && d.row < p.B && d.grow >= 0 && p0 >= 0) {
            const int32_t* bt = p.block_table + (int64_t)d.grow * p.max_pages;
            const int head0 = ((int)blockIdx.x % HGn) * HG;
            for (int j = lane; j < np; j += 32) {
                const int page = ld_relaxed_s32(bt + ((p0 + j) >> pgs));
                const int tok = ((p0 + j) & pmask) << 4;
                if (page >= 0 && (int64_t)page < p.num_pages) {
                    tma_prefetch_5d(&tmap_k, 0, tok, 0, head0, page);
                    tma_prefetch_5d(&tmap_v, 0, tok, 0, head0, page);
                }
            }
            // q rows of the unit's HG*G query heads: HG*G*256 bytes, one 128-byte line per lane
            const char* qrow = reinterpret_cast<const char*>(p.q + ((int64_t)d.grow * p.Hq + head0 * G) * D);
            for (int b = lane * 128; b < HG * G * D * 2; b += 32 * 128) prefetch_l2(qrow + b);
        }
    }
    pdl_wait();   // queue (builder), q / seq_lens (upstream), out / partials (previous step's readers)
    if (tid == 0) PKV_TRACE_STAMP(p, 1);
    if (warp == kPlanWarp) {
        // ================================================================ planner warp
        // Fused build: producer 0 derives split_offsets from seq_lens
        // (one load round trip + warp scans) and leaves the plan in shared memory; this warp --
        // off everybody's critical path -- writes this CTA's share of the queue (RowSlots, task
        // list, split_offsets, header) that the merge kernel and pkv_read_workqueue read, and
        // the outputs of rows without a task.
        if (p.fused_build) {
            named_bar_sync(kPlanBar, 64);   // producer 0 has planned (it arrives without waiting)
            const int32_t row_slots = tail.plan_row_slots;
            if (plan.split_mode == PKV_SPLIT_BALANCED) {
                plan.split_mode = PKV_SPLIT_FIXED_CHUNK;
                plan.chunk_tiles = tail.plan_chunk;
            }
            const PlanTotals tot = plan_warp_totals(plan, tail.len_s, row_slots, lane);
            for (int rs = blockIdx.x * 32 + lane; rs < tot.row_slots; rs += gridDim.x * 32) {
                int32_t tb, te;
                const RowSlot d = make_rowslot(plan, tail.so_s, tail.len_s, rs, &tb, &te);
                write_pair(plan, d, tb, te, rs, p.rowslots, p.tasks, p.tasks_cap);
            }
            if (blockIdx.x == 0) {
                for (int i = lane; i <= p.B; i += 32) p.split_offsets[i] = tail.so_s[i];
                if (lane == 0) {
                    const int64_t total = (int64_t)tot.row_slots * p.Hkv;
                    p.hdr->num_tasks = (int32_t)(total < p.tasks_cap ? total : p.tasks_cap);
                    p.hdr->max_row_splits = tot.max_n;
                    p.hdr->total_row_slots = tot.row_slots;
                    p.hdr->resolved_splits = plan.S;
                    p.hdr->chunk_tiles = plan.split_mode == PKV_SPLIT_FIXED_COUNT ? 0 : plan.chunk_tiles;
                    p.hdr->empty_tasks = (tot.row_slots - tot.sum_n) * p.Hkv;
                    if (total > p.tasks_cap) atomicOr(&p.hdr->error_word, (int32_t)PKV_DEVERR_QUEUE_OVERFLOW);
                    p.hdr->sum_seq_lens = tot.sum_seq;
                    p.hdr->build_launches = 0;
                    p.hdr->launched_build = 0;
                }
            }
        }
        if (blockIdx.x == 0 && lane == 0) {   // this launch's mark (pkv_counters.launched_*)
            p.hdr->launched_decode = 1;
            p.hdr->launched_merge = 0;
        }
        for (int i = blockIdx.x; i < p.B; i += gridDim.x) {   // rows without a task (A9)
            const int64_t gi = request_row(p.row_index, i);
            if ((p.fused_build ? tail.len_s[i] : __ldcg(p.seq_lens + gi)) > 0) continue;
            for (int e = lane; e < p.Hq * D; e += 32) {
                p.out[gi * p.Hq * D + e] = __float2half_rn(0.f);
                if (p.lse && e < p.Hq) p.lse[gi * p.Hq + e] = -INFINITY;
            }
        }
        return;
    }
    if (p.fused_build && warp == 0) {
        // Producer 0 plans for itself -- the plan is on the critical path of the first TMA load --
        // and leaves it in shared memory for the planner warp, which writes the queue.
        int32_t row_slots = spec_row_slots;
        int32_t* const err = blockIdx.x == 0 ? &p.hdr->error_word : nullptr;   // one CTA reports bad lengths
        // The first unit's block-table entries are requested together with the lengths the plan is
        // validated against: one round trip instead of two on the way to the first TMA load.
        if (!p.force_replan && (int)blockIdx.x < spec_row_slots * HGn) {
            const RowSlot d = tail.first_slot;
            const int p0 = d.tok0 >> 4;
            const int np = d.tok0 < d.tok1 ? min(((d.tok1 + 15) >> 4) - p0, (p.max_pages << pgs) - p0) : 0;
            if (d.row >= 0 && d.row < p.B && d.grow >= 0 && p0 >= 0) {
                early_row = d.grow; early_tok0 = d.tok0; early_tok1 = d.tok1;
                if (lane < np) early_mine = __ldcg(p.block_table + (int64_t)d.grow * p.max_pages + ((p0 + lane) >> pgs));
            }
        }
        if (!p.force_replan && plan_lens_unchanged(plan, p.seq_lens, tail.len_s, lane, err)) {
            plan = spec_plan;
        } else {
            __syncwarp();
            row_slots = plan_warp_prefix(plan, p.seq_lens, tail.so_s, tail.len_s, lane, (int)blockIdx.x / HGn,
                                         &tail.first_slot, err);
        }
        if (lane == 0) {
            tail.plan_row_slots = row_slots;
            tail.plan_chunk = plan.chunk_tiles;
            PKV_TRACE_STAMP(p, 8);
        }
        __syncwarp();
        named_bar_arrive(kPlanBar, 64);
        num_units = row_slots * HGn;
    }

    // ---- unit hand-out (producer 0) / pick-up (everybody else) -------------------------------
    // producer 0 reads the unit's RowSlot (one 32-byte load; the first one is issued together with
    // the header load) and publishes it on the ring; everybody else picks it up from shared memory
    auto next_unit = [&](int k) -> UnitInfo {
        const int r = k % kRing;
        UnitInfo u;
        if (warp == 0) {
            int t;
            if (k == 0 || !p.dynamic_sched) {
                t = blockIdx.x + k * gridDim.x;
            } else {
                t = 0;
                if (lane == 0) t = atomicAdd(&p.hdr->work_counter, 1) + gridDim.x;
                t = __shfl_sync(0xffffffffu, t, 0);
            }
            if (p.fused_build) {
                if (t >= num_units) t = -1;
                RowSlot d = {};
                int32_t tb, te;
                if (t >= 0 && k == 0) d = tail.first_slot;   // computed by the planner warp
                else if (t >= 0) d = make_rowslot(plan, tail.so_s, tail.len_s, t / HGn, &tb, &te);
                u.row = d.row; u.so = d.so; u.n = d.n; u.split = d.split; u.tok0 = d.tok0; u.tok1 = d.tok1;
                u.grow = d.grow; u.nlen = d.nlen;
            } else {
                const int4* rsp = reinterpret_cast<const int4*>(p.rowslots + (k == 0 ? t / HGn : min(t, max(num_units - 1, 0)) / HGn));
                const int4 a = __ldcg(rsp);
                const int4 b = __ldcg(rsp + 1);
                if (k == 0) num_units = __ldcg(&p.hdr->total_row_slots) * HGn;
                if (t >= num_units) t = -1;
                u.row = a.x; u.so = a.y; u.n = a.z; u.split = a.w; u.tok0 = b.x; u.tok1 = b.y; u.grow = b.z; u.nlen = b.w;
            }
            u.unit = t;
            if (lane == 0) {
                mbar_wait(rempty0 + 8 * r, ((k / kRing) & 1) ^ 1);
                tail.ring[r] = u;
                mbar_arrive(rfull0 + 8 * r);
            }
        } else {
            mbar_wait(rfull0 + 8 * r, (k / kRing) & 1);
            u = tail.ring[r];
            __syncwarp();
            if (lane == 0) {
                // The slot is released only after its loads have RETURNED: the store below needs
                // every field (an mbarrier arrive may otherwise overtake loads still in flight).
                sts_b32(smem_u32(&tail.sink_i[warp]),
                        (uint32_t)(u.unit + u.row + u.so + u.n + u.split + u.tok0 + u.tok1 + u.grow + u.nlen));
                mbar_arrive(rempty0 + 8 * r);
            }
        }
        return u;
    };

    if (warp < NP) {
        // ================================================================ producer warps
        // Page j of a unit is the next page of this CTA's stream of pages: it lands in stage ps,
        // in that stage's fill number whose parity is pphase.  STAGE OWNERSHIP: stage s is always
        // filled by producer s % NP and, per head, always consumed by compute warp s % WPH, so the
        // owner of a stage sees every one of its phases in order.  (A parity wait can only tell
        // adjacent phases apart: a warp that skipped a phase of a stage could pass the wait for
        // the next one while the skipped fill is still in flight.)
        uint32_t ps = 0, pphase = 0;
        const unsigned long long kv_policy = l2_policy_evict_first();
        for (int k = 0;; ++k) {
            const UnitInfo u = next_unit(k);
            if (u.unit < 0) break;
            if (k == 0 && tid == 0) PKV_TRACE_STAMP(p, 2);
            const int row = u.grow, hg = u.unit % HGn;   // the producers only need the request row
            const int tok0 = u.tok0, tok1 = u.tok1;
            if (tok0 >= tok1) continue;  // empty split: nothing is staged
            const int p0 = tok0 >> 4;
            const int np = ((tok1 + 15) >> 4) - p0;
            const int head0 = hg * HG;
            const int32_t* bt = p.block_table + (int64_t)row * p.max_pages;
            // table entries 32 blocks at a time (lane i holds the page of block c + i of the unit)
            const bool early = k == 0 && warp == 0 && row == early_row && tok0 == early_tok0 && tok1 == early_tok1;
            int mine = lane < np ? checked_page(early ? early_mine : bt[(p0 + lane) >> pgs], p.plan.flags, p.num_pages, &p.hdr->error_word) : 0;
            for (int c = 0; c < np; c += 32) {
                const int nxt = (c + 32 + lane < np)
                                    ? checked_page(bt[(p0 + c + 32 + lane) >> pgs], p.plan.flags, p.num_pages, &p.hdr->error_word) : 0;
                const int cnt = min(32, np - c);
                for (int i = 0; i < cnt; ++i) {
                    const int page = __shfl_sync(0xffffffffu, mine, i);
                    const int tok = ((p0 + c + i) & pmask) << 4;   // the block's first token inside its page
                    const uint32_t s = ps, par = pphase;
                    if (++ps == (uint32_t)kStages) { ps = 0; pphase ^= 1; }
                    if ((s % NP) != (uint32_t)warp) continue;
                    if (lane == 0) {
                        if (k == 0 && c == 0 && i == 0 && warp == 0) PKV_TRACE_STAMP(p, 3);
                        mbar_wait(empty0 + 8 * s, par ^ 1);
                        const uint32_t dst = stage_base + s * kStageBytes;
                        // box dims: (64 ch, 16 tok, D / 64 channel blocks, HG heads, 1 page)
                        mbar_arrive_expect_tx(fullk0 + 8 * s, HG * kHeadBytes);
                        tma_load_5d(dst, &tmap_k, fullk0 + 8 * s, 0, tok, 0, head0, page, kv_policy);
                        mbar_arrive_expect_tx(fullv0 + 8 * s, HG * kHeadBytes);
                        tma_load_5d(dst + HG * kHeadBytes, &tmap_v, fullv0 + 8 * s, 0, tok, 0, head0, page, kv_policy);
                    }
                }
                mine = nxt;
            }
        }
        // the last CTA to run out of units re-arms the counters for the next launch / replay
        if (warp == 0 && lane == 0) {
            PKV_TRACE_STAMP(p, 7);
            const int old = atomicAdd(&p.hdr->done_counter, 1);
            if (old == (int)gridDim.x - 1) {
                p.hdr->work_counter = 0;
                p.hdr->done_counter = 0;
            }
        }
    } else {
        // ================================================================ compute warps
        const int cw = warp - NP;            // 0..7
        const int grp = cw % NGRP;           // (head, block) group
        const int hl = grp % HG;             // head within the unit's head group
        const int h0 = (grp / HG) * GW;      // first query head of the warp's block within the KV head
        const int sub = cw / NGRP;           // which of the group's WPH warps
        const int gtid = sub * 32 + lane;    // thread index within the head's warp group
        const int g4 = lane >> 2;            // fragment "groupID"
        const int t4 = lane & 3;             // fragment "threadID_in_group"
        const int hA = 2 * t4, hB = 2 * t4 + 1;   // the two query heads (MMA N columns) this lane tracks
        // ldmatrix lane addressing inside a head's 4 KiB [2 halves][16 tok][64 ch] block
        const uint32_t k_tok = (lane & 7) + ((lane >> 3) & 1) * 8;
        const uint32_t k_sel = lane >> 4;
        const uint32_t v_tok = ((lane >> 4) << 3) + (lane & 7);
        const uint32_t v_sel = (lane >> 3) & 1;
        const uint32_t xr = lane & 7;        // swizzle: 16-byte chunk index ^= token % 8

        uint32_t cs = 0, cphase = 0;   // stage / phase parity of the unit's next page (= the producers' ps, pphase)
        for (int k = 0;; ++k) {
            const UnitInfo u = next_unit(k);
            if (u.unit < 0) break;
            const int row = u.row, orow = u.grow, hg = u.unit % HGn;
            const int so = u.so, n_i = u.n, split = u.split;
            const int kvh = hg * HG + hl;
            const int64_t slot = (int64_t)so * p.Hkv + (int64_t)kvh * n_i + split;
            const int tok0 = u.tok0, tok1 = u.tok1;
            if (tok0 >= tok1) {
                store_empty_task<G, WPH, GW>(p, &tail.cb.flag[grp], row, orow, kvh, split, n_i, slot, gtid, 1 + grp, h0);
                continue;
            }
            const int p0 = tok0 >> 4;
            const int np = ((tok1 + 15) >> 4) - p0;

            // FP8 caches (reading A28): x = (scale * k_scale[kvh]) * <q, e4m3(K)>, O = v_scale[kvh] * ...
            float sc = p.scale, sc2 = p.scale_log2, vsc = 1.f;
            if constexpr (FP8) {
                const float ksc = p.k_scale ? __ldg(p.k_scale + kvh) : 1.f;
                sc *= ksc;
                sc2 *= ksc;
                vsc = p.v_scale ? __ldg(p.v_scale + kvh) : 1.f;
            }
            // Q^T as the MMA B operand: b0 = Q[head g4][kk*16 + 2*t4 .. +1], b1 = same + 8.
            // FP8: a lane's ldmatrix word holds FOUR consecutive channels 4*t4 .. 4*t4+3 of the
            // 16-channel chunk; they stand for k = 2*t4, 2*t4+1 (a0/a1) and k = 2*t4+8, 2*t4+9
            // (a2/a3), so Q is read with the same permutation of the contraction index.
            uint32_t qb[KK][2];
            {
                const __half* qrow = p.q + ((int64_t)orow * p.Hq + kvh * G + h0 + (g4 < GW ? g4 : 0)) * D;
#pragma unroll
                for (int kk = 0; kk < KK; ++kk) {
                    const uint32_t lo = *reinterpret_cast<const uint32_t*>(qrow + kk * 16 + (FP8 ? 4 * t4 : 2 * t4));
                    const uint32_t hi = *reinterpret_cast<const uint32_t*>(qrow + kk * 16 + (FP8 ? 4 * t4 + 2 : 8 + 2 * t4));
                    qb[kk][0] = g4 < GW ? lo : 0u;
                    qb[kk][1] = g4 < GW ? hi : 0u;
                }
            }
            // Fused KV-append (+RoPE) (reading A29): q is rotated to the new token's position
            // N - 1 in registers -- the rotate-half partner of channel c < d/2 is channel c + d/2, i.e.
            // the same fragment slot of k-step kk + KK/2 -- in FP32, product by product, as the oracle.
            bool patch = false;
            int last_blk = -1, last_row = 0;
            if constexpr (APP) {
                if (p.k_new != nullptr) {
                    const int pos = u.nlen - 1;
                    patch = tok1 == u.nlen;            // this unit's range ends with the row's new token
                    last_blk = pos >> 4;
                    last_row = pos & 15;
                    if (p.rope_cos != nullptr && pos < p.rope_positions) {
                        const float* cr = p.rope_cos + (int64_t)pos * (D / 2);
                        const float* sr = p.rope_sin + (int64_t)pos * (D / 2);
#pragma unroll
                        for (int kk = 0; kk < KK / 2; ++kk) {
#pragma unroll
                            for (int hf = 0; hf < 2; ++hf) {
                                // channels c, c+1 (< d/2) of fragment slot (kk, hf); one-byte caches read Q with
                                // the permuted contraction index (see qb above)
                                const int c = kk * 16 + (FP8 ? 4 * t4 + 2 * hf : 2 * t4 + 8 * hf);
                                const float2 cs2 = __ldg(reinterpret_cast<const float2*>(cr + c));
                                const float2 sn2 = __ldg(reinterpret_cast<const float2*>(sr + c));
                                const float2 x1 = __half22float2(*reinterpret_cast<const __half2*>(&qb[kk][hf]));
                                const float2 x2 = __half22float2(*reinterpret_cast<const __half2*>(&qb[kk + KK / 2][hf]));
                                const float y1x = __fsub_rn(__fmul_rn(x1.x, cs2.x), __fmul_rn(x2.x, sn2.x));
                                const float y1y = __fsub_rn(__fmul_rn(x1.y, cs2.y), __fmul_rn(x2.y, sn2.y));
                                const float y2x = __fadd_rn(__fmul_rn(x2.x, cs2.x), __fmul_rn(x1.x, sn2.x));
                                const float y2y = __fadd_rn(__fmul_rn(x2.y, cs2.y), __fmul_rn(x1.y, sn2.y));
                                qb[kk][hf] = pack_half2(y1x, y1y);
                                qb[kk + KK / 2][hf] = pack_half2(y2x, y2y);
                            }
                        }
                    }
                }
            }
            float mA = -INFINITY, mB = -INFINITY, lA = 0.f, lB = 0.f;
            float o[KK][4];
#pragma unroll
            for (int mt = 0; mt < KK; ++mt) o[mt][0] = o[mt][1] = o[mt][2] = o[mt][3] = 0.f;

            bool first_page = true;
            // This warp's pages of the unit: those landing in the stages it owns (s % WPH == sub).
            // From an owned stage s the next owned one is s + WPH, or -- past the end of the ring --
            // stage `sub` of the next phase.  (A per-page skip loop costs > 1 us per launch.)
            int j;
            uint32_t s, par;
            {
                const uint32_t d0 = (uint32_t)(sub + WPH - (int)(cs % WPH)) % WPH;
                if (cs + d0 < (uint32_t)kStages) { j = (int)d0; s = cs + d0; par = cphase; }
                else { j = (int)((uint32_t)kStages - cs) + sub; s = (uint32_t)sub; par = cphase ^ 1; }
                const uint32_t adv = cs + (uint32_t)np;   // stream position after the unit
                cs = adv % kStages;
                cphase ^= (adv / kStages) & 1;
            }
            while (j < np) {
                const uint32_t kb = stage_base + s * kStageBytes + hl * kHeadBytes;
                const uint32_t vb = kb + HG * kHeadBytes;
                const int nvalid = tok1 - ((p0 + j) << 4);  // >= 1; >= 16 for all but the last page

                // ---- S^T = K . Q^T, two accumulation chains (channel halves)
                mbar_wait(fullk0 + 8 * s, par);
                if (k == 0 && first_page && cw == 0 && lane == 0) PKV_TRACE_STAMP(p, 4);
                first_page = false;
                if constexpr (APP) {
                    // the block that holds the row's new token: its K row comes from k_new (rotated), not
                    // from the pool -- patched into the stage here and written to the pool for later steps
                    if (patch && p0 + j == last_blk) {
                        // G = 16: the two warps of a KV head (one per block of 8 query heads) read the same
                        // stage; the first block's warp patches, its partner waits for the patch
                        if (NBK == 1 || h0 == 0) {
                            if constexpr (FP8) append_patch_q8<KVT, true>(p, kb, orow, kvh, u.nlen - 1, last_row, lane, pgs);
                            else append_patch<D, true>(p, kb, orow, kvh, u.nlen - 1, last_row, lane, pgs);
                        }
                        if constexpr (NBK > 1) named_bar_sync(kPatchBar0 + sub * HG + hl, NBK * 32);
                    }
                }
                float c0[4] = {0.f, 0.f, 0.f, 0.f}, c1[4] = {0.f, 0.f, 0.f, 0.f};
                if constexpr (FP8) {
                    // one ldmatrix.x4 = 16 tokens x 32 channels of bytes: (tok 0-7 | 8-15) x (chunk 2j | 2j+1)
#pragma unroll
                    for (int j = 0; j < KK / 2; ++j) {
                        uint32_t r0, r1, r2, r3;
                        const uint32_t chunk = (j << 1) | k_sel;
                        ldmatrix_x4(kb + k_tok * 128 + ((chunk ^ xr) << 4), r0, r1, r2, r3);
                        mma_16816(c0, cvt_bytes2_to_half2<KVT>(r0), cvt_bytes2_to_half2<KVT>(r1), cvt_bytes2_to_half2<KVT>(r0 >> 16),
                                  cvt_bytes2_to_half2<KVT>(r1 >> 16), qb[2 * j][0], qb[2 * j][1]);
                        mma_16816(c1, cvt_bytes2_to_half2<KVT>(r2), cvt_bytes2_to_half2<KVT>(r3), cvt_bytes2_to_half2<KVT>(r2 >> 16),
                                  cvt_bytes2_to_half2<KVT>(r3 >> 16), qb[2 * j + 1][0], qb[2 * j + 1][1]);
                    }
                } else {
#pragma unroll
                    for (int kk = 0; kk < KK; ++kk) {
                        uint32_t a0, a1, a2, a3;
                        const uint32_t chunk = ((kk & 3) << 1) | k_sel;
                        ldmatrix_x4(kb + (kk >> 2) * 2048 + k_tok * 128 + ((chunk ^ xr) << 4), a0, a1, a2, a3);
                        if (((kk >> 2) & 1) == 0)   // alternate 64-channel blocks between the two chains
                            mma_16816(c0, a0, a1, a2, a3, qb[kk][0], qb[kk][1]);
                        else
                            mma_16816(c1, a0, a1, a2, a3, qb[kk][0], qb[kk][1]);
                    }
                }
                // lane holds S^T[tok g4][hA], [g4][hB], [g4+8][hA], [g4+8][hB]
                float s0 = c0[0] + c1[0], s1 = c0[1] + c1[1], s2 = c0[2] + c1[2], s3 = c0[3] + c1[3];
                if (g4 >= nvalid) { s0 = -INFINITY; s1 = -INFINITY; }       // tokens past N_i (A10)
                if (g4 + 8 >= nvalid) { s2 = -INFINITY; s3 = -INFINITY; }

                // ---- online softmax: row max over the page's 16 tokens (lanes with equal t4)
                float mxA = fmaxf(s0, s2), mxB = fmaxf(s1, s3);
#pragma unroll
                for (int off = 4; off <= 16; off <<= 1) {
                    mxA = fmaxf(mxA, __shfl_xor_sync(0xffffffffu, mxA, off));
                    mxB = fmaxf(mxB, __shfl_xor_sync(0xffffffffu, mxB, off));
                }
                const float nmA = fmaxf(mA, mxA), nmB = fmaxf(mB, mxB);   // finite: the page has a valid token
                if (__any_sync(0xffffffffu, (nmA != mA) | (nmB != mB))) {
                    const float alA = ex2_approx((mA - nmA) * sc2);  // m = -inf -> 0
                    const float alB = ex2_approx((mB - nmB) * sc2);
                    lA *= alA;
                    lB *= alB;
#pragma unroll
                    for (int mt = 0; mt < KK; ++mt) {
                        o[mt][0] *= alA; o[mt][2] *= alA;
                        o[mt][1] *= alB; o[mt][3] *= alB;
                    }
                    mA = nmA;
                    mB = nmB;
                }
                const float offA = mA * sc2, offB = mB * sc2;
                const float p0f = ex2_approx(fmaf(s0, sc2, -offA));
                const float p1f = ex2_approx(fmaf(s1, sc2, -offB));
                const float p2f = ex2_approx(fmaf(s2, sc2, -offA));
                const float p3f = ex2_approx(fmaf(s3, sc2, -offB));
                lA += p0f + p2f;   // lane-partial sums; reduced across lanes at unit end
                lB += p1f + p3f;
                // P^T as the MMA B operand: transpose the two 8x8 (token x head) blocks
                const uint32_t pb0 = movmatrix_trans(pack_half2(p0f, p1f));
                const uint32_t pb1 = movmatrix_trans(pack_half2(p2f, p3f));

                // ---- O^T += V^T . P^T
                mbar_wait(fullv0 + 8 * s, par);
                if constexpr (APP) {
                    if (patch && p0 + j == last_blk) {
                        if (NBK == 1 || h0 == 0) {
                            if constexpr (FP8) append_patch_q8<KVT, false>(p, vb, orow, kvh, u.nlen - 1, last_row, lane, pgs);
                            else append_patch<D, false>(p, vb, orow, kvh, u.nlen - 1, last_row, lane, pgs);
                        }
                        if constexpr (NBK > 1) named_bar_sync(kPatchBar0 + sub * HG + hl, NBK * 32);
                    }
                }
                uint32_t vdep = 0;   // a word of every V fragment (see the stage release below)
                if constexpr (FP8) {
                    // ldmatrix.trans moves 16-bit units, i.e. PAIRS of channels: a lane gets tokens
                    // 2*t4, 2*t4+1 of the channel pair (2*g4, 2*g4+1) of a 16-channel chunk.  Byte
                    // permutes split the pair: MMA row g4 is channel 16*mt + 2*g4, row g4+8 is channel
                    // 16*mt + 2*g4 + 1 (the epilogue stores with the same map).
#pragma unroll
                    for (int j = 0; j < KK / 2; ++j) {
                        uint32_t r0, r1, r2, r3;
                        const uint32_t chunk = (j << 1) | k_sel;
                        ldmatrix_x4_trans(vb + k_tok * 128 + ((chunk ^ xr) << 4), r0, r1, r2, r3);
                        mma_16816(o[2 * j], cvt_bytes2_to_half2<KVT>(__byte_perm(r0, 0, 0x0020)), cvt_bytes2_to_half2<KVT>(__byte_perm(r0, 0, 0x0031)),
                                  cvt_bytes2_to_half2<KVT>(__byte_perm(r1, 0, 0x0020)), cvt_bytes2_to_half2<KVT>(__byte_perm(r1, 0, 0x0031)), pb0, pb1);
                        mma_16816(o[2 * j + 1], cvt_bytes2_to_half2<KVT>(__byte_perm(r2, 0, 0x0020)), cvt_bytes2_to_half2<KVT>(__byte_perm(r2, 0, 0x0031)),
                                  cvt_bytes2_to_half2<KVT>(__byte_perm(r3, 0, 0x0020)), cvt_bytes2_to_half2<KVT>(__byte_perm(r3, 0, 0x0031)), pb0, pb1);
                        vdep ^= r0 ^ r1 ^ r2 ^ r3;
                    }
                } else {
#pragma unroll
                    for (int mt = 0; mt < KK; ++mt) {
                        uint32_t a0, a1, a2, a3;
                        const uint32_t chunk = ((mt & 3) << 1) | v_sel;
                        ldmatrix_x4_trans(vb + (mt >> 2) * 2048 + v_tok * 128 + ((chunk ^ xr) << 4), a0, a1, a2, a3);
                        mma_16816(o[mt], a0, a1, a2, a3, pb0, pb1);
                        vdep ^= a3;
                    }
                }
                __syncwarp();
                if (lane == 0) {
                    // This head's part of the stage is consumed -- but only once the LAST ldmatrix
                    // has returned its data.  ptxas schedules the arrive right behind the issue of
                    // that ldmatrix, ahead of the HMMAs that wait for it, and the arrive can
                    // overtake the load when the SM's memory pipe is backed up: the producer then
                    // refills the stage under the load (seen as stale V rows in channels 112..127,
                    // DESIGN.md "stage release").  The store needs a word of every V fragment, so
                    // it cannot issue before all eight ldmatrix have completed, and a
                    // release-arrive cannot move above a store of its own thread.
                    sts_b32(smem_u32(&tail.sink_f[cw]), vdep);
                    mbar_arrive(empty0 + 8 * s);
                }
                if (s + WPH < (uint32_t)kStages) { s += WPH; j += WPH; }
                else { j += (int)((uint32_t)kStages - s) + sub; s = (uint32_t)sub; par ^= 1; }
            }
            if (k == 0 && cw == 0 && lane == 0) PKV_TRACE_STAMP(p, 5);

            // ---- warp state -> combine buffer row cw
#pragma unroll
            for (int off = 4; off <= 16; off <<= 1) {
                lA += __shfl_xor_sync(0xffffffffu, lA, off);
                lB += __shfl_xor_sync(0xffffffffu, lB, off);
            }
            // channels of accumulator rows g4 and g4 + 8 inside an m-tile of 16 (FP8: see the V loop)
            const int cA = FP8 ? 2 * g4 : g4, cB = FP8 ? 2 * g4 + 1 : g4 + 8;
            if constexpr (WPH == 1) {
                // The warp owns the whole task: its state goes from the MMA accumulators straight
                // to the task's slot (or to `out`), no shared-memory round trip.  Per store
                // instruction the 8 lanes of a column write 32 contiguous bytes.
                if (hA < GW) {
                    const bool hasB = hB < GW;   // G = 1: column B is padding
                    const int64_t hrow = (int64_t)orow * p.Hq + kvh * G + h0 + hA;
                    if (n_i <= 1) {
                        const float iA = vsc / lA, iB = hasB ? vsc / lB : 0.f;
                        __half* oA = p.out + hrow * D;
                        __half* oB = oA + D;
#pragma unroll
                        for (int mt = 0; mt < KK; ++mt) {
                            oA[mt * 16 + cA] = __float2half_rn(o[mt][0] * iA);
                            oA[mt * 16 + cB] = __float2half_rn(o[mt][2] * iA);
                            if (hasB) {
                                oB[mt * 16 + cA] = __float2half_rn(o[mt][1] * iB);
                                oB[mt * 16 + cB] = __float2half_rn(o[mt][3] * iB);
                            }
                        }
                        if (p.lse && g4 == 0) {
                            p.lse[hrow] = mA * sc + logf(lA);
                            if (hasB) p.lse[hrow + 1] = mB * sc + logf(lB);
                        }
                    } else {
                        float* aA = p.part_acc + (slot * G + h0 + hA) * D;
                        float* aB = aA + D;
#pragma unroll
                        for (int mt = 0; mt < KK; ++mt) {
                            aA[mt * 16 + cA] = o[mt][0] * vsc;
                            aA[mt * 16 + cB] = o[mt][2] * vsc;
                            if (hasB) {
                                aB[mt * 16 + cA] = o[mt][1] * vsc;
                                aB[mt * 16 + cB] = o[mt][3] * vsc;
                            }
                        }
                        if (g4 == 0) {
                            p.part_m[slot * G + h0 + hA] = mA * sc;
                            p.part_l[slot * G + h0 + hA] = lA;
                            if (hasB) {
                                p.part_m[slot * G + h0 + hB] = mB * sc;
                                p.part_l[slot * G + h0 + hB] = lB;
                            }
                        }
                    }
                }
                if (n_i > 1 && p.merge_mode == PKV_MERGE_FUSED)
                    fused_complete<G, 1>(p, &tail.cb.flag[cw], row, orow, kvh, split, n_i, slot, lane, 1 + grp, NBK);
            } else {
                if (hA < GW) {
                    const bool hasB = hB < GW;   // G = 1: column B is padding
#pragma unroll
                    for (int mt = 0; mt < KK; ++mt) {
                        tail.cb.acc[cw][hA][mt * 16 + cA] = o[mt][0] * vsc;
                        tail.cb.acc[cw][hA][mt * 16 + cB] = o[mt][2] * vsc;
                        if (hasB) {
                            tail.cb.acc[cw][hB][mt * 16 + cA] = o[mt][1] * vsc;
                            tail.cb.acc[cw][hB][mt * 16 + cB] = o[mt][3] * vsc;
                        }
                    }
                    if (g4 == 0) {
                        tail.cb.m[cw][hA] = mA; tail.cb.l[cw][hA] = lA;
                        if (hasB) { tail.cb.m[cw][hB] = mB; tail.cb.l[cw][hB] = lB; }
                    }
                }
                group_sync<WPH>(1 + grp);
                finalize_task<G, WPH, kComputeWarps, GW, D>(p, tail.cb, grp, NGRP, row, orow, kvh, split, n_i, slot, gtid, 1 + grp, h0, sc, sc2);
            }
            if (k == 0 && cw == 0 && lane == 0) PKV_TRACE_STAMP(p, 6);
        }
    }
}

template <int G, int HG, int D, int KVT, bool APP = false>
cudaError_t launch_one(const DecodeParams& p, int grid, const CUtensorMap& mk, const CUtensorMap& mv,
                       cudaStream_t stream) {
    constexpr int smem = stages_for<G, HG, D, KVT != 0>() * stage_bytes_for(HG, D, KVT != 0) + (int)sizeof(SmemTail<G / blocks_for(G), D>) + 1024;
    constexpr int threads = (producers_for(HG) + kComputeWarps + 1) * 32;
    // The dynamic shared-memory opt-in is a per-device (per-context) attribute of the kernel: one
    // flag per device ordinal, set on the first launch there (races only repeat the call).
    static bool attr_set[64] = {};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64 || !attr_set[dev]) {
        e = cudaFuncSetAttribute(pkv_decode_tma_kernel<G, HG, D, KVT, APP>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
        if (dev >= 0 && dev < 64) attr_set[dev] = true;
    }
    return launch_pdl(!(p.plan.flags & PKV_FLAG_NO_PDL), pkv_decode_tma_kernel<G, HG, D, KVT, APP>, dim3(grid), dim3(threads),
                      (size_t)smem, stream, p, mk, mv);
}

}  // namespace

template <int PART>
cudaError_t launch_decode_tma_part(const DecodeParams& p, int G, int HG, int D, int kvt, bool app, int grid, const CUtensorMap& mk,
                                   const CUtensorMap& mv, cudaStream_t stream);

// The 147 instantiations are compiled as kTmaParts translation units of this one source
// (-DPKV_TMA_PART=k, see build.py): part k defines launch_decode_tma_part<k>, which launches the
// kernel if the requested instantiation belongs to it and returns cudaErrorNotSupported otherwise;
// part 0 also holds the dispatcher.
#ifndef PKV_TMA_PART
#define PKV_TMA_PART 0
#endif

#define PKV_CASE(GG, HH, DD, KK, AA) \
    if (G == GG && HG == HH && D == DD && kvt == KK && app == AA) return launch_one<GG, HH, DD, KK, AA>(p, grid, mk, mv, stream);
#define PKV_CASE_HG(GG, DD, KK, AA) PKV_CASE(GG, 8, DD, KK, AA) PKV_CASE(GG, 4, DD, KK, AA) PKV_CASE(GG, 2, DD, KK, AA) PKV_CASE(GG, 1, DD, KK, AA)
#define PKV_CASE_HG4(GG, DD, KK, AA) PKV_CASE(GG, 4, DD, KK, AA) PKV_CASE(GG, 2, DD, KK, AA) PKV_CASE(GG, 1, DD, KK, AA)

template <>
cudaError_t launch_decode_tma_part<PKV_TMA_PART>(const DecodeParams& p, int G, int HG, int D, int kvt, bool app, int grid,
                                                 const CUtensorMap& mk, const CUtensorMap& mv, cudaStream_t stream) {
#if PKV_TMA_PART == 0      // the paper's shapes: FP16, d = 128, G = 4 and 8
    PKV_CASE_HG(4, 128, 0, false) PKV_CASE_HG(8, 128, 0, false)
#elif PKV_TMA_PART == 1    // G = 1, 2 and 16 (two blocks of 8 query heads: at most 4 heads per CTA)
    PKV_CASE_HG(2, 128, 0, false) PKV_CASE_HG(1, 128, 0, false) PKV_CASE_HG4(16, 128, 0, false)
#elif PKV_TMA_PART == 2    // head dimensions 64 and 256 (d = 256: at most 4 heads per CTA, a stage of 8 would be 128 KiB)
    PKV_CASE_HG(4, 64, 0, false) PKV_CASE_HG(8, 64, 0, false) PKV_CASE_HG4(4, 256, 0, false) PKV_CASE_HG4(8, 256, 0, false)
#elif PKV_TMA_PART == 3    // FP8 (E4M3) caches
    PKV_CASE_HG(4, 128, 1, false) PKV_CASE_HG(8, 128, 1, false)
#elif PKV_TMA_PART == 4    // INT8 caches
    PKV_CASE_HG(4, 128, 2, false) PKV_CASE_HG(8, 128, 2, false)
#elif PKV_TMA_PART == 5    // fused KV-append + RoPE, G = 4 and 8
    PKV_CASE_HG(4, 128, 0, true) PKV_CASE_HG(8, 128, 0, true)
#elif PKV_TMA_PART == 6    // fused KV-append + RoPE, G = 1 and 2
    PKV_CASE_HG(2, 128, 0, true) PKV_CASE_HG(1, 128, 0, true)
#elif PKV_TMA_PART == 7    // FP8 (E4M3) caches, G = 1, 2 and 16
    PKV_CASE_HG(2, 128, 1, false) PKV_CASE_HG(1, 128, 1, false) PKV_CASE_HG4(16, 128, 1, false)
#elif PKV_TMA_PART == 8    // INT8 caches, G = 1, 2 and 16
    PKV_CASE_HG(2, 128, 2, false) PKV_CASE_HG(1, 128, 2, false) PKV_CASE_HG4(16, 128, 2, false)
#elif PKV_TMA_PART == 9    // d = 64, G = 1, 2 and 16
    PKV_CASE_HG(2, 64, 0, false) PKV_CASE_HG(1, 64, 0, false) PKV_CASE_HG4(16, 64, 0, false)
#elif PKV_TMA_PART == 10   // d = 256, G = 1, 2 and 16
    PKV_CASE_HG4(2, 256, 0, false) PKV_CASE_HG4(1, 256, 0, false) PKV_CASE_HG4(16, 256, 0, false)
#elif PKV_TMA_PART == 11   // fused KV-append on FP8 (E4M3) caches, G = 4 and 8
    PKV_CASE_HG(4, 128, 1, true) PKV_CASE_HG(8, 128, 1, true)
#elif PKV_TMA_PART == 12   // fused KV-append on INT8 caches, G = 4 and 8
    PKV_CASE_HG(4, 128, 2, true) PKV_CASE_HG(8, 128, 2, true)
#elif PKV_TMA_PART == 13   // fused KV-append on FP8 (E4M3) caches, G = 1 and 2
    PKV_CASE_HG(2, 128, 1, true) PKV_CASE_HG(1, 128, 1, true)
#elif PKV_TMA_PART == 14   // fused KV-append on INT8 caches, G = 1 and 2
    PKV_CASE_HG(2, 128, 2, true) PKV_CASE_HG(1, 128, 2, true)
#elif PKV_TMA_PART == 15   // fused KV-append, G = 16 (FP16, FP8 and INT8 caches)
    PKV_CASE_HG4(16, 128, 0, true) PKV_CASE_HG4(16, 128, 1, true) PKV_CASE_HG4(16, 128, 2, true)
#endif
    return cudaErrorNotSupported;
}
#undef PKV_CASE_HG4
#undef PKV_CASE_HG
#undef PKV_CASE

#if PKV_TMA_PART == 0
int decode_tma_stage_bytes(int HG, int D, bool fp8) { return stage_bytes_for(HG, D, fp8); }

cudaError_t launch_decode_tma(const DecodeParams& p, int G, int HG, int D, int kvt, int grid, const void* tmap_k,
                              const void* tmap_v, cudaStream_t stream) {
    if (grid <= 0) return cudaSuccess;
    const CUtensorMap& mk = *reinterpret_cast<const CUtensorMap*>(tmap_k);
    const CUtensorMap& mv = *reinterpret_cast<const CUtensorMap*>(tmap_v);
    const bool app = p.k_new != nullptr;
    cudaError_t e = launch_decode_tma_part<0>(p, G, HG, D, kvt, app, grid, mk, mv, stream);
    if (e == cudaErrorNotSupported) e = launch_decode_tma_part<1>(p, G, HG, D, kvt, app, grid, mk, mv, stream);
    if (e == cudaErrorNotSupported) e = launch_decode_tma_part<2>(p, G, HG, D, kvt, app, grid, mk, mv, stream);
    if (e == cudaErrorNotSupported) e = launch_decode_tma_part<3>(p, G, HG, D, kvt, app, grid, mk, mv, stream);
    if (e == cudaErrorNotSupported) e = launch_decode_tma_part<4>(p, G, HG, D, kvt, app, grid, mk, mv, stream);
    if (e == cudaErrorNotSupported) e = launch_decode_tma_part<5>(p, G, HG, D, kvt, app, grid, mk, mv, stream);
    if (e == cudaErrorNotSupported) e = launch_decode_tma_part<6>(p, G, HG, D, kvt, app, grid, mk, mv, stream);
    if (e == cudaErrorNotSupported) e = launch_decode_tma_part<7>(p, G, HG, D, kvt, app, grid, mk, mv, stream);
    if (e == cudaErrorNotSupported) e = launch_decode_tma_part<8>(p, G, HG, D, kvt, app, grid, mk, mv, stream);
    if (e == cudaErrorNotSupported) e = launch_decode_tma_part<9>(p, G, HG, D, kvt, app, grid, mk, mv, stream);
    if (e == cudaErrorNotSupported) e = launch_decode_tma_part<10>(p, G, HG, D, kvt, app, grid, mk, mv, stream);
    if (e == cudaErrorNotSupported) e = launch_decode_tma_part<11>(p, G, HG, D, kvt, app, grid, mk, mv, stream);
    if (e == cudaErrorNotSupported) e = launch_decode_tma_part<12>(p, G, HG, D, kvt, app, grid, mk, mv, stream);
    if (e == cudaErrorNotSupported) e = launch_decode_tma_part<13>(p, G, HG, D, kvt, app, grid, mk, mv, stream);
    if (e == cudaErrorNotSupported) e = launch_decode_tma_part<14>(p, G, HG, D, kvt, app, grid, mk, mv, stream);
    if (e == cudaErrorNotSupported) e = launch_decode_tma_part<15>(p, G, HG, D, kvt, app, grid, mk, mv, stream);
    return e == cudaErrorNotSupported ? cudaErrorInvalidValue : e;
}
#endif

}  // namespace pkv
