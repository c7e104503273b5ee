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
    int32_t B, Hkv, S, tile_tokens, split_mode, chunk_tiles, route;
};

// One CTA (blockDim.x = 128 .. 1024, a multiple of 32).
// Phase 1: per-row slot counts and their exclusive prefix sum (split_offsets).
// Phase 2: one thread per (row, split) pair rs = tid, tid + blockDim.x, ...: the row is found by
// binary search in split_offsets; the thread writes the pair's RowSlot and its Hkv task entries
// at so*Hkv + g*n + s, so the list comes out in (row, kvh, split) order.
__global__ void __launch_bounds__(kBuildThreadsMax) pkv_build_workqueue_kernel(const BuildArgs a) {
    __shared__ int32_t warp_sums[32];
    __shared__ int32_t carry_s;
    __shared__ int32_t max_n_s, empties_s;
    __shared__ unsigned long long sum_seq_s;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nthreads = blockDim.x, nwarps = nthreads >> 5;
    pdl_launch_dependents();
    if (tid == 0) {
        carry_s = 0;
        max_n_s = 0;
        empties_s = 0;
        sum_seq_s = 0ull;
    }
    pdl_wait();   // the queue may still be read by the previous step's kernels
    if (tid == 0) a.split_offsets[0] = 0;
    __syncthreads();
    for (int base = 0; base < a.B; base += nthreads) {
        const int i = base + tid;
        int32_t slots = 0, N = 0;
        if (i < a.B) {
            N = max(a.seq_lens[i], 0);
            const RowSplits r = row_splits(N, a.tile_tokens, a.split_mode, a.S, a.chunk_tiles);
            slots = a.route == PKV_ROUTE_WORKQUEUE ? r.n : a.S;
        }
        // inclusive warp scan, then scan of warp totals
        int32_t v = slots;
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            const int32_t u = __shfl_up_sync(0xffffffffu, v, off);
            if (lane >= off) v += u;
        }
        if (lane == 31) warp_sums[warp] = v;
        __syncthreads();
        if (warp == 0) {
            int32_t w = lane < nwarps ? warp_sums[lane] : 0;
#pragma unroll
            for (int off = 1; off < 32; off <<= 1) {
                const int32_t u = __shfl_up_sync(0xffffffffu, w, off);
                if (lane >= off) w += u;
            }
            warp_sums[lane] = w;  // inclusive
        }
        __syncthreads();
        const int32_t incl = carry_s + (warp > 0 ? warp_sums[warp - 1] : 0) + v;
        if (i < a.B) {
            a.split_offsets[i + 1] = incl;
            atomicMax(&max_n_s, slots);
            atomicAdd(&sum_seq_s, (unsigned long long)N);
        }
        __syncthreads();
        if (tid == nthreads - 1) carry_s = incl;
        __syncthreads();
    }
    for (int i = tid; i < a.B * a.Hkv; i += nthreads) a.fuse_counters[i] = 0;
    __threadfence_block();
    __syncthreads();

    const int32_t row_slots = carry_s;
    const int64_t total = (int64_t)row_slots * a.Hkv;
    int32_t my_empties = 0;
    for (int32_t rs = tid; rs < row_slots; rs += nthreads) {
        // largest row with split_offsets[row] <= rs
        int lo = 0, hi = a.B - 1;
        while (lo < hi) {
            const int mid = (lo + hi + 1) >> 1;
            if (a.split_offsets[mid] <= rs) lo = mid; else hi = mid - 1;
        }
        const int row = lo;
        const int32_t so = a.split_offsets[row];
        const int32_t slots = a.split_offsets[row + 1] - so;
        const int32_t s = rs - so;
        const int32_t N = max(a.seq_lens[row], 0);
        const RowSplits r = row_splits(N, a.tile_tokens, a.split_mode, a.S, a.chunk_tiles);
        int32_t tb = 0, te = 0;
        if (r.T > 0) {
            const int64_t b = (int64_t)s * r.c, e = (int64_t)(s + 1) * r.c;
            tb = (int32_t)(b < r.T ? b : r.T);
            te = (int32_t)(e < r.T ? e : r.T);
        }
        if (tb >= te) my_empties += a.Hkv;
        RowSlot d;
        d.row = row; d.so = so; d.n = slots; d.split = s;
        d.tok0 = tb * a.tile_tokens;
        d.tok1 = min(te * a.tile_tokens, N);
        d.pad_[0] = d.pad_[1] = 0;
        a.rowslots[rs] = d;
        for (int g = 0; g < a.Hkv; ++g) {
            const int64_t idx = (int64_t)so * a.Hkv + (int64_t)g * slots + s;
            if (idx < a.tasks_cap) {
                pkv_task t;
                t.row = row; t.kvh = g; t.split = s; t.t_begin = tb; t.t_end = te;
                a.tasks[idx] = t;
            }
        }
    }
    if (my_empties) atomicAdd(&empties_s, my_empties);
    __syncthreads();
    if (tid == 0) {
        QueueHeader h;
        h.num_tasks = (int32_t)(total < a.tasks_cap ? total : a.tasks_cap);
        h.max_row_splits = max_n_s;
        h.total_row_slots = row_slots;
        h.resolved_splits = a.S;
        h.empty_tasks = empties_s;
        h.work_counter = 0;
        h.done_counter = 0;
        h.error_word = total > a.tasks_cap ? 1 : 0;
        h.sum_seq_lens = (int64_t)sum_seq_s;
        h.pad_[0] = h.pad_[1] = h.pad_[2] = 0;
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
    a.B = shape.B; a.Hkv = shape.Hkv; a.S = rp.S; a.tile_tokens = rp.tile_tokens;
    a.split_mode = rp.split_mode; a.chunk_tiles = rp.chunk_tiles; a.route = rp.route;
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
