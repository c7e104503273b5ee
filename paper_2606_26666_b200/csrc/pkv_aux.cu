// pkv_aux.cu -- the two small kernels around the decode kernel:
//   * device workqueue builder: split-bound policy from the true row lengths
//     and the compact task list in canonical order (A6-A8);
//   * segmented merge of split states.
#include "pkv_device.cuh"

namespace pkv {

namespace {

constexpr int kBuildThreadsMax = 1024;
constexpr int kBuildWarpPlanRows = 512;   // up to this many rows the builder uses the decode kernel's warp planner

struct BuildArgs {
    const int32_t* seq_lens;
    QueueHeader* hdr;
    int32_t* split_offsets;
    int32_t* fuse_counters;
    RowSlot* rowslots;
    pkv_task* tasks;
    int64_t tasks_cap;
    PlanArgs plan;
};

// One CTA (blockDim.x = 128 .. 1024).  Phase 1: plan_scan -> split_offsets.  Phase 2: one thread
// per (row, split) pair writes the pair's RowSlot and its Hkv task entries (pkv_device.cuh).
__global__ void __launch_bounds__(kBuildThreadsMax) pkv_build_workqueue_kernel(const BuildArgs a) {
    __shared__ PlanScratch sc;
    __shared__ int32_t so_s[kBuildWarpPlanRows + 1], len_s[kBuildWarpPlanRows];
    __shared__ RowSlot unused_first;
    __shared__ PlanTotals tot_s;
    __shared__ int32_t chunk_s;
    const int tid = threadIdx.x, nthreads = blockDim.x;
    pdl_launch_dependents();
    pdl_wait();   // the queue may still be read by the previous step's kernels
    PlanArgs plan = a.plan;   // BALANCED: the planner resolves the batch-wide chunk into this copy
    PlanTotals tot;
    const int32_t* so = a.split_offsets;
    const int32_t* lens = a.seq_lens;
    if (plan.B <= kBuildWarpPlanRows) {
        // the decode kernel's own planner (plan_warp_prefix / plan_warp_totals): one warp plans
        // into shared memory, everybody writes the queue -- so that this entry point and the
        // fused build run (and the tests of either exercise) the same code
        if (tid < 32) {
            const int32_t rs = plan_warp_prefix(plan, a.seq_lens, so_s, len_s, tid, -1, &unused_first, &a.hdr->error_word);
            const PlanTotals t = plan_warp_totals(plan, len_s, rs, tid);
            if (tid == 0) { tot_s = t; chunk_s = plan.chunk_tiles; }
        }
        __syncthreads();
        tot = tot_s;
        if (plan.split_mode == PKV_SPLIT_BALANCED) {
            plan.split_mode = PKV_SPLIT_FIXED_CHUNK;
            plan.chunk_tiles = chunk_s;
        }
        for (int i = tid; i <= plan.B; i += nthreads) a.split_offsets[i] = so_s[i];
        so = so_s;
        lens = len_s;
    } else {
        tot = plan_scan(plan, a.seq_lens, a.split_offsets, nullptr, sc, &a.hdr->error_word);
    }
    for (int i = tid; i < a.plan.B * a.plan.Hkv; i += nthreads) a.fuse_counters[i] = 0;
    __threadfence_block();
    __syncthreads();
    const int64_t total = (int64_t)tot.row_slots * a.plan.Hkv;
    for (int32_t rs = tid; rs < tot.row_slots; rs += nthreads) {
        int32_t tb, te;
        const RowSlot d = make_rowslot(plan, so, lens, rs, &tb, &te);
        write_pair(plan, d, tb, te, rs, a.rowslots, a.tasks, a.tasks_cap);
    }
    if (tid == 0) {   // field by field: error_word is sticky and only ever OR-ed into
        QueueHeader* h = a.hdr;
        h->num_tasks = (int32_t)(total < a.tasks_cap ? total : a.tasks_cap);
        h->max_row_splits = tot.max_n;
        h->total_row_slots = tot.row_slots;
        h->resolved_splits = a.plan.S;
        h->empty_tasks = (tot.row_slots - tot.sum_n) * a.plan.Hkv;   // rect route; 0 on the workqueue route
        h->work_counter = 0;
        h->done_counter = 0;
        if (total > a.tasks_cap) atomicOr(&h->error_word, (int32_t)PKV_DEVERR_QUEUE_OVERFLOW);
        h->sum_seq_lens = tot.sum_seq;
        h->build_launches = 1;
        h->chunk_tiles = plan.split_mode == PKV_SPLIT_FIXED_COUNT ? 0 : plan.chunk_tiles;
        h->launched_build = 1;
        h->launched_decode = 0;
        h->launched_merge = 0;
    }
}

// One CTA of NW warps per (row, query head, channel slice); a slice is 128 / CS channels (CS = 1, 2
// or 4), a row of d channels has d * CS / 128 of them.  A state's slice is read by 32 / CS lanes (16 bytes each), so one load instruction of
// a warp covers CS states; every lane issues the loads of kMergeBatch states (m, l and its piece
// of acc) before any arithmetic, so a row of up to NW * kMergeBatch * CS splits is ONE round trip
// to L2, and folds them into an online state (M, L, A) -- the merge of PAPER.md:60-61 is
// associative, so the lane states of a warp (shuffles) and the NW warp states (shared memory)
// combine exactly the same way, in a fixed order (deterministic).  Rows with at most one slot were
// written directly by the decode kernel.  Slices spread a single long row (B = 1: 32 (row, head)
// pairs of 128 .. 148 splits) over 128 small CTAs instead of 32 large ones: four times the SMs
// pull the states out of L2, and 4-warp CTAs fit beside a resident decode CTA, so they are in
// place -- guess made, waiting -- when the decode grid finishes.  NW and CS are chosen at launch.
struct MergeState {
    float M, L;
    float4 A;
};
__device__ __forceinline__ void merge_combine(MergeState& a, float M2, float L2, const float4& A2) {
    const float nM = fmaxf(a.M, M2);
    if (nM == -INFINITY) return;                              // both neutral
    const float w1 = ex2_approx((a.M - nM) * kLog2e);         // exp2(-inf) = 0
    const float w2 = ex2_approx((M2 - nM) * kLog2e);
    a.L = fmaf(w2, L2, w1 * a.L);
    a.A.x = fmaf(w2, A2.x, w1 * a.A.x); a.A.y = fmaf(w2, A2.y, w1 * a.A.y);
    a.A.z = fmaf(w2, A2.z, w1 * a.A.z); a.A.w = fmaf(w2, A2.w, w1 * a.A.w);
    a.M = nM;
}

template <int G, int NW, int CS, int MINB>
__global__ void __launch_bounds__(NW * 32, MINB) pkv_merge_kernel(const DecodeParams p) {
    constexpr int NB = kMergeBatch;
    constexpr int LPS = 32 / CS;          // lanes per state
    __shared__ float4 sA[NW][LPS];
    __shared__ float sM[NW], sL[NW];
    const int nsl = p.d / (LPS * 4);      // slices of LPS * 4 channels per (row, head): d * CS / 128
    const int slice = blockIdx.x % nsl, rh = blockIdx.x / nsl;
    const int row = rh / p.Hq, h = rh % p.Hq;
    const int kvh = h / G, hh = h % G;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int sub = lane / LPS, cl = lane % LPS;
    const int ch = slice * (LPS * 4) + cl * 4;   // this lane's four channels
    if (blockIdx.x == 0 && threadIdx.x == 0) PKV_TRACE_STAMP_MERGE(p, 0);
    pdl_launch_dependents();
    // A guess at the row's slot range, read (race-tolerant) before the decode grid has finished:
    // merge CTAs are resident long before their wait returns, and from one decode step to the
    // next the ranges rarely move.  After the wait the first batch of states is requested from
    // the guessed range TOGETHER with the real split_offsets -- one round trip instead of two --
    // and thrown away if the guess was wrong.  The guess is only used if it lies inside the
    // partial-state buffers.
    const int so_g = ld_relaxed_s32(p.split_offsets + row);
    const int n_g = ld_relaxed_s32(p.split_offsets + row + 1) - so_g;
    const bool guess = p.tasks_cap > 0 && so_g >= 0 && n_g > 1 && ((int64_t)so_g + (int64_t)n_g) * p.Hkv <= p.tasks_cap;
    pdl_wait();
    if (blockIdx.x == 0 && threadIdx.x == 0) PKV_TRACE_STAMP_MERGE(p, 1);
    if (blockIdx.x == 0 && threadIdx.x == 0 && p.hdr != nullptr) p.hdr->launched_merge = 1;   // this launch's mark
    const int so = __ldcg(p.split_offsets + row);
    const int n = __ldcg(p.split_offsets + row + 1) - so;
    const int orow = request_row(p.row_index, row);   // loaded with the offsets: no extra round trip
    // batch b of this warp: states (b * NB * NW + j * NW + warp) * CS + sub, j = 0 .. NB-1
    auto load_batch = [&](int64_t base_, int n_, int b, float (&mv)[NB], float (&lv)[NB], float4 (&av)[NB]) {
#pragma unroll
        for (int j = 0; j < NB; ++j) {
            const int s_ = ((b * NB + j) * NW + warp) * CS + sub;
            const bool ok = s_ < n_;
            const int64_t r = (base_ + (ok ? s_ : 0)) * G + hh;
            mv[j] = ok ? __ldcg(p.part_m + r) : -INFINITY;
            lv[j] = ok ? __ldcg(p.part_l + r) : 0.f;
            av[j] = ok ? __ldcg(reinterpret_cast<const float4*>(p.part_acc + r * p.d + ch))
                       : make_float4(0.f, 0.f, 0.f, 0.f);
        }
    };
    float mv[NB], lv[NB];
    float4 av[NB];
    if (guess) load_batch((int64_t)so_g * p.Hkv + (int64_t)kvh * n_g, n_g, 0, mv, lv, av);
    if (n <= 1 && p.hdr != nullptr) return;   // library path: decode already produced out/lse
    const bool hit = guess && so == so_g && n == n_g;
    const int64_t base = (int64_t)so * p.Hkv + (int64_t)kvh * n;
    MergeState st;
    st.M = -INFINITY; st.L = 0.f; st.A = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int b = 0; b * NB * NW * CS < n; ++b) {
        if (!(hit && b == 0)) load_batch(base, n, b, mv, lv, av);
        float mb = mv[0];
#pragma unroll
        for (int j = 1; j < NB; ++j) mb = fmaxf(mb, mv[j]);
        const float nM = fmaxf(st.M, mb);
        if (nM == -INFINITY) continue;        // only neutral states so far
        const float al = ex2_approx((st.M - nM) * kLog2e);   // M = -inf -> 0
        st.L *= al;
        st.A.x *= al; st.A.y *= al; st.A.z *= al; st.A.w *= al;
#pragma unroll
        for (int j = 0; j < NB; ++j) {
            const float w = ex2_approx((mv[j] - nM) * kLog2e);   // exp2(-inf) = 0
            st.L = fmaf(w, lv[j], st.L);
            st.A.x = fmaf(w, av[j].x, st.A.x); st.A.y = fmaf(w, av[j].y, st.A.y);
            st.A.z = fmaf(w, av[j].z, st.A.z); st.A.w = fmaf(w, av[j].w, st.A.w);
        }
        st.M = nM;
    }
    // the CS lane groups of the warp hold different states of the same channels
#pragma unroll
    for (int off = LPS; off < 32; off <<= 1) {
        const float M2 = __shfl_xor_sync(0xffffffffu, st.M, off), L2 = __shfl_xor_sync(0xffffffffu, st.L, off);
        float4 A2;
        A2.x = __shfl_xor_sync(0xffffffffu, st.A.x, off); A2.y = __shfl_xor_sync(0xffffffffu, st.A.y, off);
        A2.z = __shfl_xor_sync(0xffffffffu, st.A.z, off); A2.w = __shfl_xor_sync(0xffffffffu, st.A.w, off);
        // the lower lane group's state goes first on both sides: identical results in all groups
        if (lane & off) {
            MergeState t; t.M = M2; t.L = L2; t.A = A2;
            merge_combine(t, st.M, st.L, st.A);
            st = t;
        } else {
            merge_combine(st, M2, L2, A2);
        }
    }
    if (sub == 0) sA[warp][cl] = st.A;
    if (lane == 0) { sM[warp] = st.M; sL[warp] = st.L; }
    __syncthreads();
    if (warp == 0 && sub == 0) {
        float Mf = sM[0];
#pragma unroll
        for (int w = 1; w < NW; ++w) Mf = fmaxf(Mf, sM[w]);
        float Ls = 0.f;
        float4 As = make_float4(0.f, 0.f, 0.f, 0.f);
        if (Mf != -INFINITY) {
#pragma unroll
            for (int w = 0; w < NW; ++w) {
                const float wt = ex2_approx((sM[w] - Mf) * kLog2e);
                const float4 a = sA[w][cl];
                Ls = fmaf(wt, sL[w], Ls);
                As.x = fmaf(wt, a.x, As.x); As.y = fmaf(wt, a.y, As.y);
                As.z = fmaf(wt, a.z, As.z); As.w = fmaf(wt, a.w, As.w);
            }
        }
        merge_store(p, (int64_t)orow * p.Hq + h, ch, slice == 0 && cl == 0, Mf, Ls, As);
        if (blockIdx.x == 0 && lane == 0) PKV_TRACE_STAMP_MERGE(p, 2);
    }
}

// Pipelined host-buffer step (pkv_decode_host_pipelined).  The step's launches are enqueued BEFORE the
// host has its inputs; this kernel is the first of them and the gate: one CTA that
//   1. lets its dependents go at once (the decode CTAs become resident, plan speculatively on the
//      previous step's lengths -- re-validated after their dependency wait -- and prefetch),
//   2. gate = true: polls the flag word of the pinned, device-mapped staging image until the host has
//      released step `seq` (one PCIe read per poll by one thread), or until `timeout_ns` have passed --
//      then it records `expired = seq` and goes on, so a stream that nobody releases is blocked for a
//      bounded time only (the step then runs on stale inputs and the host discards its result),
//   3. fetches the step's small inputs -- lengths, q, changed block-table rows -- from the image over
//      the host link into the device scratch (same layout: a segment is (offset, 16-byte chunks));
//      system-scope volatile loads: the CPU wrote these bytes after the launch was enqueued,
//   4. tells the host that it has finished reading the image (`staged = seq`).
__global__ void __launch_bounds__(kStageThreads) pkv_stage_kernel(const unsigned char* __restrict__ src, unsigned char* __restrict__ dst,
                                                                  const StageSegs segs, volatile uint32_t* words, uint32_t seq, bool gate,
                                                                  unsigned long long timeout_ns) {
    pdl_launch_dependents();
    if (gate) {
        if (threadIdx.x == 0) {
            unsigned long long t0, t1;
            asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t0));
            while ((int32_t)(words[kPipeFlagWord] - seq) < 0) {
                asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t1));
                if (t1 - t0 > timeout_ns) {
                    words[kPipeExpiredWord] = seq;
                    break;
                }
            }
        }
        __syncthreads();
    }
#pragma unroll
    for (int k = 0; k < kMaxStageSegs; ++k) {
        if (k >= segs.n) break;
        const size_t base = segs.off[k];
        // four loads in flight per thread: 64 KiB cross the host link in one round trip, not four
        for (uint32_t i0 = threadIdx.x; i0 < segs.chunks[k]; i0 += 4 * kStageThreads) {
            uint4 v[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const uint32_t i = i0 + u * kStageThreads;
                if (i < segs.chunks[k])
                    asm volatile("ld.volatile.global.v4.u32 {%0, %1, %2, %3}, [%4];"
                                 : "=r"(v[u].x), "=r"(v[u].y), "=r"(v[u].z), "=r"(v[u].w)
                                 : "l"(src + base + 16 * (size_t)i));
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const uint32_t i = i0 + u * kStageThreads;
                if (i < segs.chunks[k]) *reinterpret_cast<uint4*>(dst + base + 16 * (size_t)i) = v[u];
            }
        }
    }
    __syncthreads();     // every load of the image has returned: its value has gone into the store behind it
    // no fence: `staged` publishes nothing, it only says that the image is no longer being read
    if (threadIdx.x == 0) words[kPipeStagedWord] = seq;
}

// Last launch of a pipelined step: resident early (programmatic launch), it waits for everything before
// it in the stream -- the merge's (or the decode's) stores to the pinned out_host included -- and
// writes the step's number into the image's `done` word, which the host is spinning on.
__global__ void __launch_bounds__(kSignalThreads) pkv_signal_kernel(volatile uint32_t* words, uint32_t seq, const uint4* out_dev, uint4* out_host,
                                                                    uint32_t out_chunks) {
    pdl_launch_dependents();
    pdl_wait();
    // the step's result, from device memory to the pinned out_host (out_chunks 16-byte pieces; 0: the
    // kernels wrote it there themselves)
    for (uint32_t i = threadIdx.x; i < out_chunks; i += kSignalThreads) out_host[i] = out_dev[i];
    __syncthreads();
    if (threadIdx.x == 0 && words != nullptr) {      // (no words: pkv_decode_host, which synchronises the stream instead)
        __threadfence_system();
        words[kPipeDoneWord] = seq;
    }
}

}  // namespace

cudaError_t launch_stage(const void* src_mapped, void* dst, const StageSegs& segs, uint32_t* words_mapped, uint32_t seq, bool gate,
                         unsigned long long timeout_ns, cudaStream_t stream) {
    // a plain launch: whatever is ahead of it in the stream (the previous step) has finished when it starts
    pkv_stage_kernel<<<1, kStageThreads, 0, stream>>>(static_cast<const unsigned char*>(src_mapped), static_cast<unsigned char*>(dst), segs,
                                                      words_mapped, seq, gate, timeout_ns);
    return cudaGetLastError();
}

cudaError_t launch_signal(uint32_t* words_mapped, uint32_t seq, bool pdl, const void* out_dev, void* out_host_mapped, size_t out_bytes,
                          cudaStream_t stream) {
    return launch_pdl(pdl, pkv_signal_kernel, dim3(1), dim3(kSignalThreads), 0, stream, (volatile uint32_t*)words_mapped, seq,
                      static_cast<const uint4*>(out_dev), static_cast<uint4*>(out_host_mapped), (uint32_t)(out_bytes / 16));
}

cudaError_t launch_builder(const pkv_shape& shape, const Resolved& rp, const int32_t* seq_lens_dev,
                           const int32_t* row_index, QueueHeader* hdr, int32_t* split_offsets, int32_t* fuse_counters, RowSlot* rowslots,
                           pkv_task* tasks, int64_t tasks_cap, cudaStream_t stream) {
    BuildArgs a;
    a.seq_lens = seq_lens_dev;
    a.hdr = hdr;
    a.split_offsets = split_offsets;
    a.fuse_counters = fuse_counters;
    a.rowslots = rowslots;
    a.tasks = tasks;
    a.tasks_cap = tasks_cap;
    a.plan = make_plan_args(shape, rp);
    a.plan.row_index = row_index;
    // one thread per (row, split) pair if that fits in a CTA, 128..1024 threads
    const int64_t want = (int64_t)shape.B * rp.S;
    int threads = 128;
    while (threads < kBuildThreadsMax && threads < want) threads <<= 1;
    return launch_pdl(!(rp.flags & PKV_FLAG_NO_PDL), pkv_build_workqueue_kernel, dim3(1), dim3(threads), 0, stream, a);
}

cudaError_t launch_merge(const DecodeParams& p, int G, cudaStream_t stream) {
    const int pairs = p.B * p.Hq;
    if (pairs <= 0) return cudaSuccess;
    const bool pdl = !(p.plan.flags & PKV_FLAG_NO_PDL);
    // Warps per CTA (NW) and channel slices (CS).  A warp covers 8 * CS splits per round trip, and
    // small CTAs start (and finish) sooner, so: as few warps as cover the row's splits in one round
    // when the split count is known on the host (FIXED_COUNT: at most S; measured on config 2,
    // S = 16: 2 warps 25.9 us per step, 4 warps 26.0, 16 warps 26.9); else by batch size -- 16 warps
    // while there is at most one (row, head) pair per SM, 8 warps up to 1024 pairs (49.6 vs 50.7 us
    // on config 3), 4 warps, six CTAs per SM, beyond (config 5).
    // Slices when rows can hold more than 32 splits and the CTAs still fit the machine in one wave
    // (B * Hq * 4 <= 160, i.e. a single long row): 128 CTAs of 8 warps pull one row's 128 .. 148
    // states per head out of L2 instead of 32 CTAs of 16 warps (config 2, whole step, S = 147:
    // 23.4 vs 24.5 us; S = 128: 23.4 vs 23.6; 4-warp CTAs and 2 slices are slower, r02 sweep).
    int nw, cs = 1;
    const bool known = p.plan.split_mode == PKV_SPLIT_FIXED_COUNT && p.plan.S > 0;
    const int n_max = known ? p.plan.S : kMaxSplits;
    if (n_max > 32 && pairs * (p.d * 4 / 128) <= 160) {
        cs = 4;
        nw = 8;
    } else if (known) {
        nw = n_max <= 16 ? 2 : (n_max <= 32 ? 4 : (n_max <= 64 ? 8 : 16));
    } else {
        nw = pairs <= 148 ? 16 : (pairs <= 1024 ? 8 : 4);
    }
    if (p.d == 64 && cs == 1) cs = 2;     // a 64-channel row is half a warp: two states per load instruction
    const int grid = pairs * (p.d * cs / 128);
#define PKV_MERGE_CASE(GG, NWW, CSS, MB) \
    if (G == GG && nw == NWW && cs == CSS)  \
        return launch_pdl(pdl, pkv_merge_kernel<GG, NWW, CSS, MB>, dim3(grid), dim3(NWW * 32), 0, stream, p);
#define PKV_MERGE_G(GG) \
    PKV_MERGE_CASE(GG, 2, 1, 1) PKV_MERGE_CASE(GG, 4, 1, 6) PKV_MERGE_CASE(GG, 8, 1, 1) PKV_MERGE_CASE(GG, 16, 1, 1) \
    PKV_MERGE_CASE(GG, 2, 2, 1) PKV_MERGE_CASE(GG, 4, 2, 1) PKV_MERGE_CASE(GG, 8, 2, 1) PKV_MERGE_CASE(GG, 16, 2, 1) \
    PKV_MERGE_CASE(GG, 2, 4, 1) PKV_MERGE_CASE(GG, 4, 4, 1) PKV_MERGE_CASE(GG, 8, 4, 1) PKV_MERGE_CASE(GG, 16, 4, 1)
    PKV_MERGE_G(4) PKV_MERGE_G(8) PKV_MERGE_G(2) PKV_MERGE_G(1) PKV_MERGE_G(16)
#undef PKV_MERGE_G
#undef PKV_MERGE_CASE
    return cudaErrorInvalidValue;
}

}  // namespace pkv
