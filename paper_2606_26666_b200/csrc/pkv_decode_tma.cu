// pkv_decode_tma.cu -- PKV_KERNEL_TMA_MMA: the B200 decode kernel.
//
// Persistent, warp-specialised CTA, one per SM (PAPER.md:42 maps one CTA to one (request, KV
// head, split) work item; here a resident CTA walks many such tasks -- DESIGN.md A20):
//
//   warp 0 (producer)    takes tasks (static stride or an atomic counter), walks the task's
//                        slice of the block table (PAPER.md:50 page accessor) 32 entries at a
//                        time, and for every page issues ONE TMA box for K and one for V: the
//                        page's 16 tokens x 128 channels of the task's KV head, 4 KiB each,
//                        128-byte swizzled, into a ring of kStages 8 KiB stages guarded by
//                        full/empty mbarriers.  It runs ahead across task boundaries, so the
//                        ring never drains between tasks.
//   warps 1..8 (compute) page j of a task belongs to warp j % 8.  Per page:
//                        S^T[16 tok x 8 heads] = K[16 x 128] . Q^T      8 HMMA m16n8k16
//                        exact online softmax in FP32, P -> FP16
//                        O^T[128 x 8 heads]  += V^T[128 x 16] . P^T     8 HMMA m16n8k16
//                        Tokens sit on the MMA M axis and the G <= 8 grouped query heads
//                         on the N = 8 axis, so G = 8 fills the tile and G = 4
//                        half of it; K is read with ldmatrix, V with ldmatrix.trans, P^T is
//                        produced from the S^T accumulator layout with movmatrix.
//   task end             the 8 warp states are combined through shared memory and stored as
//                        the split's partial state, or directly as FP16 output when the row
//                        has a single split (pkv_device.cuh finalize_task).
#include <cuda.h>

#include "pkv_device.cuh"

namespace pkv {

namespace {

constexpr int kComputeWarps = 8;
constexpr int kThreadsTma = (1 + kComputeWarps) * 32;
constexpr int kComputeThreads = kComputeWarps * 32;
constexpr int kStageBytes = 8192;   // K 4096 | V 4096
constexpr int kRing = 4;            // task-id ring between producer and compute warps
constexpr int kBarCompute = 1;      // named barrier of the compute warps

template <int G>
struct SmemTail {
    CombineBuf<G, kComputeWarps> cb;
    unsigned long long full_bar[32];   // kStages <= 32
    unsigned long long empty_bar[32];
    unsigned long long ring_full[kRing];
    unsigned long long ring_empty[kRing];
    int task_ring[kRing];
};

template <int G>
__host__ __device__ constexpr int stages_for() {
    // 227 KiB per CTA, minus the tail, minus 1 KiB alignment slack
    return (int)((232448 - 1024 - (int)sizeof(SmemTail<G>)) / kStageBytes) > 32
               ? 32
               : (int)((232448 - 1024 - (int)sizeof(SmemTail<G>)) / kStageBytes);
}

template <int G>
__global__ void __launch_bounds__(kThreadsTma, 1)
    pkv_decode_tma_kernel(const DecodeParams p, const __grid_constant__ CUtensorMap tmap_k,
                          const __grid_constant__ CUtensorMap tmap_v) {
    constexpr int kStages = stages_for<G>();
    extern __shared__ unsigned char smem_raw[];
    // 128-byte swizzle: every 2 KiB half-box must start on a 1024-byte boundary
    unsigned char* smem = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    SmemTail<G>& tail = *reinterpret_cast<SmemTail<G>*>(smem + (size_t)kStages * kStageBytes);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const uint32_t stage_base = smem_u32(smem);
    const uint32_t full0 = smem_u32(&tail.full_bar[0]);
    const uint32_t empty0 = smem_u32(&tail.empty_bar[0]);
    const uint32_t rfull0 = smem_u32(&tail.ring_full[0]);
    const uint32_t rempty0 = smem_u32(&tail.ring_empty[0]);

    if (tid == 0) {
        for (int s = 0; s < kStages; ++s) {
            mbar_init(full0 + 8 * s, 1);
            mbar_init(empty0 + 8 * s, 1);
        }
        for (int r = 0; r < kRing; ++r) {
            mbar_init(rfull0 + 8 * r, 1);
            mbar_init(rempty0 + 8 * r, kComputeWarps);
        }
        mbar_fence_init();
        tma_prefetch_desc(&tmap_k);
        tma_prefetch_desc(&tmap_v);
    }
    zero_empty_rows(p);
    __syncthreads();

    const int num_tasks = p.hdr->num_tasks;

    if (warp == 0) {
        // ================================================================ producer warp
        uint32_t seq = 0;  // pages issued by this CTA so far
        for (int k = 0;; ++k) {
            int t;
            if (k == 0 || !p.dynamic_sched) {
                t = blockIdx.x + k * gridDim.x;
            } else {
                t = 0;
                if (lane == 0) t = atomicAdd(&p.hdr->work_counter, 1) + gridDim.x;
                t = __shfl_sync(0xffffffffu, t, 0);
            }
            if (t >= num_tasks) t = -1;
            const int r = k % kRing;
            if (lane == 0) {
                mbar_wait(rempty0 + 8 * r, ((k / kRing) & 1) ^ 1);
                tail.task_ring[r] = t;
                mbar_arrive(rfull0 + 8 * r);
            }
            if (t < 0) break;
            const pkv_task task = p.tasks[t];
            const int N = p.seq_lens[task.row];
            const int tok0 = task.t_begin * p.tile_tokens;
            const int tok1 = min(task.t_end * p.tile_tokens, N);
            if (tok0 >= tok1) continue;  // empty split: nothing is staged
            const int p0 = tok0 >> 4;
            const int np = ((tok1 + 15) >> 4) - p0;
            const int32_t* bt = p.block_table + (int64_t)task.row * p.max_pages + p0;
            int mine = (lane < np) ? bt[lane] : 0;
            for (int c = 0; c < np; c += 32) {
                // next 32 table entries are fetched while this batch of boxes is issued
                const int nxt = (c + 32 + lane < np) ? bt[c + 32 + lane] : 0;
                const int cnt = min(32, np - c);
                for (int j = 0; j < cnt; ++j) {
                    const int page = __shfl_sync(0xffffffffu, mine, j);
                    if (lane == 0) {
                        const uint32_t s = seq % kStages;
                        const uint32_t use = seq / kStages;
                        mbar_wait(empty0 + 8 * s, (use & 1) ^ 1);
                        const uint32_t fb = full0 + 8 * s;
                        const uint32_t dst = stage_base + s * kStageBytes;
                        mbar_arrive_expect_tx(fb, kStageBytes);
                        if (p.tma_rank == 0) {
                            // dims: (64 ch, 16 tok, 2 ch-halves, head, page)
                            tma_load_5d(dst, &tmap_k, fb, 0, 0, 0, task.kvh, page);
                            tma_load_5d(dst + 4096, &tmap_v, fb, 0, 0, 0, task.kvh, page);
                        } else {
                            // dims: (128 ch, 16 tok, head, page) or (128 ch, head, 16 tok, page); box 64 ch wide
                            const int c1 = p.tma_rank == 1 ? 0 : task.kvh;
                            const int c2 = p.tma_rank == 1 ? task.kvh : 0;
                            tma_load_4d(dst, &tmap_k, fb, 0, c1, c2, page);
                            tma_load_4d(dst + 2048, &tmap_k, fb, 64, c1, c2, page);
                            tma_load_4d(dst + 4096, &tmap_v, fb, 0, c1, c2, page);
                            tma_load_4d(dst + 6144, &tmap_v, fb, 64, c1, c2, page);
                        }
                    }
                    ++seq;
                }
                mine = nxt;
            }
        }
        // the last CTA to run out of tasks re-arms the counters for the next launch / replay
        if (lane == 0) {
            const int old = atomicAdd(&p.hdr->done_counter, 1);
            if (old == (int)gridDim.x - 1) {
                p.hdr->work_counter = 0;
                p.hdr->done_counter = 0;
            }
        }
    } else {
        // ================================================================ compute warps
        const int cw = warp - 1;             // 0..7
        const int ctid = tid - 32;           // 0..255
        const int g4 = lane >> 2;            // fragment "groupID"
        const int t4 = lane & 3;             // fragment "threadID_in_group"
        const int hA = 2 * t4, hB = 2 * t4 + 1;   // the two heads (MMA N columns) this lane tracks
        // ldmatrix lane addressing inside a stage (see header comment)
        const uint32_t k_tok = (lane & 7) + ((lane >> 3) & 1) * 8;
        const uint32_t k_sel = lane >> 4;
        const uint32_t v_tok = ((lane >> 4) << 3) + (lane & 7);
        const uint32_t v_sel = (lane >> 3) & 1;
        const uint32_t xr = lane & 7;        // swizzle: 16-byte chunk index ^= token % 8

        uint32_t seq_base = 0;
        for (int k = 0;; ++k) {
            const int r = k % kRing;
            mbar_wait(rfull0 + 8 * r, (k / kRing) & 1);
            const int t = tail.task_ring[r];
            __syncwarp();
            if (lane == 0) mbar_arrive(rempty0 + 8 * r);
            if (t < 0) break;
            const pkv_task task = p.tasks[t];
            const int row = task.row, kvh = task.kvh;
            const int N = p.seq_lens[row];
            const int so = p.split_offsets[row];
            const int n_i = p.split_offsets[row + 1] - so;
            const int64_t slot = (int64_t)so * p.Hkv + (int64_t)kvh * n_i + task.split;
            const int tok0 = task.t_begin * p.tile_tokens;
            const int tok1 = min(task.t_end * p.tile_tokens, N);
            if (tok0 >= tok1) {
                store_empty_task<G>(p, row, kvh, n_i, slot, ctid, kComputeThreads);
                continue;
            }
            const int p0 = tok0 >> 4;
            const int np = ((tok1 + 15) >> 4) - p0;

            // Q^T as the MMA B operand: b0 = Q[head g4][kk*16 + 2*t4 .. +1], b1 = same + 8
            uint32_t qb[8][2];
            {
                const __half* qrow = p.q + ((int64_t)row * p.Hq + kvh * G + (g4 < G ? g4 : 0)) * kD;
#pragma unroll
                for (int kk = 0; kk < 8; ++kk) {
                    const uint32_t lo = *reinterpret_cast<const uint32_t*>(qrow + kk * 16 + 2 * t4);
                    const uint32_t hi = *reinterpret_cast<const uint32_t*>(qrow + kk * 16 + 8 + 2 * t4);
                    qb[kk][0] = g4 < G ? lo : 0u;
                    qb[kk][1] = g4 < G ? hi : 0u;
                }
            }
            float mA = -INFINITY, mB = -INFINITY, lA = 0.f, lB = 0.f;
            float o[8][4];
#pragma unroll
            for (int mt = 0; mt < 8; ++mt) o[mt][0] = o[mt][1] = o[mt][2] = o[mt][3] = 0.f;

            for (int j = cw; j < np; j += kComputeWarps) {
                const uint32_t sq = seq_base + j;
                const uint32_t s = sq % kStages;
                mbar_wait(full0 + 8 * s, (sq / kStages) & 1);
                const uint32_t kb = stage_base + s * kStageBytes;
                const uint32_t vb = kb + 4096;
                const int nvalid = tok1 - ((p0 + j) << 4);  // >= 1; >= 16 for all but the last page

                // ---- S^T = K . Q^T, two accumulation chains (channel halves)
                float c0[4] = {0.f, 0.f, 0.f, 0.f}, c1[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
                for (int kk = 0; kk < 8; ++kk) {
                    uint32_t a0, a1, a2, a3;
                    const uint32_t chunk = ((kk & 3) << 1) | k_sel;
                    ldmatrix_x4(kb + (kk >> 2) * 2048 + k_tok * 128 + ((chunk ^ xr) << 4), a0, a1, a2, a3);
                    if (kk < 4)
                        mma_16816(c0, a0, a1, a2, a3, qb[kk][0], qb[kk][1]);
                    else
                        mma_16816(c1, a0, a1, a2, a3, qb[kk][0], qb[kk][1]);
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
                    const float alA = ex2_approx((mA - nmA) * p.scale_log2);  // m = -inf -> 0
                    const float alB = ex2_approx((mB - nmB) * p.scale_log2);
                    lA *= alA;
                    lB *= alB;
#pragma unroll
                    for (int mt = 0; mt < 8; ++mt) {
                        o[mt][0] *= alA; o[mt][2] *= alA;
                        o[mt][1] *= alB; o[mt][3] *= alB;
                    }
                    mA = nmA;
                    mB = nmB;
                }
                const float offA = mA * p.scale_log2, offB = mB * p.scale_log2;
                const float p0f = ex2_approx(fmaf(s0, p.scale_log2, -offA));
                const float p1f = ex2_approx(fmaf(s1, p.scale_log2, -offB));
                const float p2f = ex2_approx(fmaf(s2, p.scale_log2, -offA));
                const float p3f = ex2_approx(fmaf(s3, p.scale_log2, -offB));
                lA += p0f + p2f;   // lane-partial sums; reduced across lanes at task end
                lB += p1f + p3f;
                // P^T as the MMA B operand: transpose the two 8x8 (token x head) blocks
                const uint32_t pb0 = movmatrix_trans(pack_half2(p0f, p1f));
                const uint32_t pb1 = movmatrix_trans(pack_half2(p2f, p3f));

                // ---- O^T += V^T . P^T
#pragma unroll
                for (int mt = 0; mt < 8; ++mt) {
                    uint32_t a0, a1, a2, a3;
                    const uint32_t chunk = ((mt & 3) << 1) | v_sel;
                    ldmatrix_x4_trans(vb + (mt >> 2) * 2048 + v_tok * 128 + ((chunk ^ xr) << 4), a0, a1, a2, a3);
                    mma_16816(o[mt], a0, a1, a2, a3, pb0, pb1);
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(empty0 + 8 * s);   // stage may be refilled
            }
            seq_base += np;

            // ---- warp state -> combine buffer
#pragma unroll
            for (int off = 4; off <= 16; off <<= 1) {
                lA += __shfl_xor_sync(0xffffffffu, lA, off);
                lB += __shfl_xor_sync(0xffffffffu, lB, off);
            }
            if (hA < G) {
#pragma unroll
                for (int mt = 0; mt < 8; ++mt) {
                    tail.cb.acc[cw][hA][mt * 16 + g4] = o[mt][0];
                    tail.cb.acc[cw][hB][mt * 16 + g4] = o[mt][1];
                    tail.cb.acc[cw][hA][mt * 16 + g4 + 8] = o[mt][2];
                    tail.cb.acc[cw][hB][mt * 16 + g4 + 8] = o[mt][3];
                }
                if (g4 == 0) {
                    tail.cb.m[cw][hA] = mA; tail.cb.m[cw][hB] = mB;
                    tail.cb.l[cw][hA] = lA; tail.cb.l[cw][hB] = lB;
                }
            }
            named_bar_sync(kBarCompute, kComputeThreads);
            finalize_task<G, kComputeWarps>(p, tail.cb, row, kvh, task.split, n_i, slot, ctid, kComputeThreads,
                                            kBarCompute);
        }
    }
}

}  // namespace

int decode_tma_smem_bytes(int G) {
    return G == 4 ? stages_for<4>() * kStageBytes + (int)sizeof(SmemTail<4>) + 1024
                  : stages_for<8>() * kStageBytes + (int)sizeof(SmemTail<8>) + 1024;
}

cudaError_t launch_decode_tma(const DecodeParams& p, int G, int grid, const void* tmap_k, const void* tmap_v,
                              cudaStream_t stream) {
    if (grid <= 0) return cudaSuccess;
    const int smem = decode_tma_smem_bytes(G);
    const CUtensorMap& mk = *reinterpret_cast<const CUtensorMap*>(tmap_k);
    const CUtensorMap& mv = *reinterpret_cast<const CUtensorMap*>(tmap_v);
    cudaError_t e;
    if (G == 4) {
        e = cudaFuncSetAttribute(pkv_decode_tma_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
        pkv_decode_tma_kernel<4><<<grid, kThreadsTma, smem, stream>>>(p, mk, mv);
    } else {
        e = cudaFuncSetAttribute(pkv_decode_tma_kernel<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
        pkv_decode_tma_kernel<8><<<grid, kThreadsTma, smem, stream>>>(p, mk, mv);
    }
    return cudaGetLastError();
}

}  // namespace pkv
