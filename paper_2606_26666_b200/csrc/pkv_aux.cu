// pkv_aux.cu -- the two small kernels around the decode kernel:
//   * device workqueue builder: split-bound policy from the true row lengths
//     and the compact task list in canonical order (A6-A8);
//   * segmented merge of split states.
#include "pkv_device.cuh"

namespace pkv {

namespace {

constexpr int kBuildThreadsMax = 1024;

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
    const int tid = threadIdx.x, nthreads = blockDim.x;
    pdl_launch_dependents();
    pdl_wait();   // the queue may still be read by the previous step's kernels
    const PlanTotals tot = plan_scan(a.plan, a.seq_lens, a.split_offsets, nullptr, sc);
    for (int i = tid; i < a.plan.B * a.plan.Hkv; i += nthreads) a.fuse_counters[i] = 0;
    __threadfence_block();
    __syncthreads();
    const int64_t total = (int64_t)tot.row_slots * a.plan.Hkv;
    for (int32_t rs = tid; rs < tot.row_slots; rs += nthreads) {
        int32_t tb, te;
        const RowSlot d = make_rowslot(a.plan, a.split_offsets, a.seq_lens, rs, &tb, &te);
        write_pair(a.plan, d, tb, te, rs, a.rowslots, a.tasks, a.tasks_cap);
    }
    if (tid == 0) {
        QueueHeader h;
        h.num_tasks = (int32_t)(total < a.tasks_cap ? total : a.tasks_cap);
        h.max_row_splits = tot.max_n;
        h.total_row_slots = tot.row_slots;
        h.resolved_splits = a.plan.S;
        h.empty_tasks = (tot.row_slots - tot.sum_n) * a.plan.Hkv;   // rect route; 0 on the workqueue route
        h.work_counter = 0;
        h.done_counter = 0;
        h.error_word = total > a.tasks_cap ? 1 : 0;
        h.sum_seq_lens = tot.sum_seq;
        h.build_launches = 1;
        h.pad32_ = 0;
        h.pad_[0] = h.pad_[1] = 0;
        *a.hdr = h;
    }
}

// One CTA of 4 warps per (row, query head): warp k computes the interleaved partial P_k of
// pkv_device.cuh's merge arithmetic, warp 0 combines the four in order.  Rows with at most one
// slot were written directly by the decode kernel.
template <int G>
__global__ void __launch_bounds__(128) pkv_merge_kernel(const DecodeParams p) {
    __shared__ float4 sA[4][32];
    __shared__ float sL[4];
    const int row = blockIdx.x / p.Hq, h = blockIdx.x % p.Hq;
    const int kvh = h / G, hh = h % G;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    pdl_launch_dependents();
    pdl_wait();
    const int so = p.split_offsets[row];
    const int n = p.split_offsets[row + 1] - so;
    if (n <= 1 && p.hdr != nullptr) return;   // library path: decode already produced out/lse
    const int64_t base = (int64_t)so * p.Hkv + (int64_t)kvh * n;
    const float M = merge_row_max<G>(p, base, n, hh, lane);
    float L[1];
    float4 A[1];
    merge_accumulate<G, 1>(p, base, n, hh, M, warp, 4, lane, L, A);
    sA[warp][lane] = A[0];
    if (lane == 0) sL[warp] = L[0];
    __syncthreads();
    if (warp == 0) {
        const float Ls = ((sL[0] + sL[1]) + sL[2]) + sL[3];
        float4 As;
        As.x = ((sA[0][lane].x + sA[1][lane].x) + sA[2][lane].x) + sA[3][lane].x;
        As.y = ((sA[0][lane].y + sA[1][lane].y) + sA[2][lane].y) + sA[3][lane].y;
        As.z = ((sA[0][lane].z + sA[1][lane].z) + sA[2][lane].z) + sA[3][lane].z;
        As.w = ((sA[0][lane].w + sA[1][lane].w) + sA[2][lane].w) + sA[3][lane].w;
        merge_store(p, (int64_t)row * p.Hq + h, lane, M, Ls, As);
    }
}

}  // namespace

cudaError_t launch_builder(const pkv_shape& shape, const Resolved& rp, const int32_t* seq_lens_dev,
                           QueueHeader* hdr, int32_t* split_offsets, int32_t* fuse_counters, RowSlot* rowslots,
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
    // one thread per (row, split) pair if that fits in a CTA, 128..1024 threads
    const int64_t want = (int64_t)shape.B * rp.S;
    int threads = 128;
    while (threads < kBuildThreadsMax && threads < want) threads <<= 1;
    return launch_pdl(pkv_build_workqueue_kernel, dim3(1), dim3(threads), 0, stream, a);
}

cudaError_t launch_merge(const DecodeParams& p, int G, cudaStream_t stream) {
    const int grid = p.B * p.Hq;
    if (grid <= 0) return cudaSuccess;
    if (G == 4) return launch_pdl(pkv_merge_kernel<4>, dim3(grid), dim3(128), 0, stream, p);
    return launch_pdl(pkv_merge_kernel<8>, dim3(grid), dim3(128), 0, stream, p);
}

}  // namespace pkv
