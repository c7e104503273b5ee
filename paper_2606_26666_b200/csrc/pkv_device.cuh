// pkv_device.cuh -- device-side declarations shared by the CUDA translation units of libpkv:
// kernel parameter block, PTX wrappers (mbarrier, TMA, ldmatrix, HMMA), and the task epilogue
// (partial-state store, direct output, fused merge) used by both decode kernels.
#pragma once

#include <cuda_fp16.h>
#include <cuda_runtime.h>

#include "pkv_common.h"

namespace pkv {

constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;

struct DecodeParams {
    const __half* q;            // [B, Hq, d]
    const __half* k_cache;      // raw pointers (SIMT kernel; the TMA kernel uses tensor maps)
    const __half* v_cache;
    const int32_t* block_table; // [B, max_pages]
    const int32_t* seq_lens;    // [B]
    const pkv_task* tasks;
    const int32_t* split_offsets; // [B+1]
    QueueHeader* hdr;
    __half* out;                // [B, Hq, d]
    float* lse;                 // [B, Hq] or nullptr
    float* part_m;              // [slots, G]
    float* part_l;              // [slots, G]
    float* part_acc;            // [slots, G, d]
    int32_t* fuse_counters;     // [B*Hkv]
    int64_t stride_page, stride_token, stride_head; // elements
    int32_t B, Hq, Hkv, max_pages, tile_tokens, merge_mode;
    int32_t tma_rank;           // tensor-map mode: 0 = rank 5, one box per (page, head); 1, 2 = rank 4, two boxes
    int32_t dynamic_sched;      // 1: tasks handed out by an atomic counter
    float scale;                // x = scale * <q, k>
    float scale_log2;           // scale * log2(e)
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
__device__ __forceinline__ void named_bar_sync(int id, int nthreads) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

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
__device__ __forceinline__ void tma_load_5d(uint32_t dst, const void* tmap, uint32_t bar, int c0, int c1,
                                            int c2, int c3, int c4) {
    asm volatile(
        "cp.async.bulk.tensor.5d.shared::cluster.global.tile.mbarrier::complete_tx::bytes "
        "[%0], [%1, {%3, %4, %5, %6, %7}], [%2];" ::"r"(dst),
        "l"(tmap), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4)
        : "memory");
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
__device__ __forceinline__ uint32_t pack_half2(float lo, float hi) {
    __half2 h = __floats2half2_rn(lo, hi);
    return *reinterpret_cast<uint32_t*>(&h);
}

// ------------------------------------------------------------------ merge of split states

// Exact merge of the n states of (row, kvh) for head-in-group `hh`, channel
// `dd`.  States live at slots slot_base .. slot_base+n-1.  One thread per (hh, dd); the
// summation order (s ascending) is the same in the separate and the fused merge.
template <int G>
__device__ __forceinline__ void merge_one(const DecodeParams& p, int64_t slot_base, int n, int row, int kvh,
                                          int hh, int dd) {
    float M = -INFINITY;
#pragma unroll 8
    for (int s = 0; s < n; ++s) M = fmaxf(M, p.part_m[(slot_base + s) * G + hh]);
    const int64_t o = ((int64_t)row * p.Hq + kvh * G + hh);
    if (M == -INFINITY) {  // no state or only neutral states (A9)
        p.out[o * kD + dd] = __float2half_rn(0.f);
        if (p.lse && dd == 0) p.lse[o] = -INFINITY;
        return;
    }
    float L = 0.f, A = 0.f;
#pragma unroll 8
    for (int s = 0; s < n; ++s) {
        const float ms = p.part_m[(slot_base + s) * G + hh];
        const float w = ex2_approx((ms - M) * kLog2e);  // exp2(-inf) = 0: neutral states drop out
        L += w * p.part_l[(slot_base + s) * G + hh];
        A += w * p.part_acc[((slot_base + s) * G + hh) * kD + dd];
    }
    p.out[o * kD + dd] = __float2half_rn(A / L);
    if (p.lse && dd == 0) p.lse[o] = M + logf(L);
}

// ------------------------------------------------------------------ task epilogue

// Shared-memory combine buffer of one CTA: the NW compute warps each leave the state of their
// share of the task's tokens here; m in raw-dot units (x = scale * raw).
constexpr int kAccStride = 132;  // floats per (warp, head) row of comb_acc; 132 % 32 = 4 spreads banks
template <int G, int NW>
struct CombineBuf {
    float acc[NW][G][kAccStride];
    float m[NW][8];
    float l[NW][8];
    int flag;
};

// Writes an empty task's result (rect route): neutral partial state, or zeros when
// the row has a single slot (direct output).
template <int G>
__device__ __forceinline__ void store_empty_task(const DecodeParams& p, int row, int kvh, int n_i, int64_t slot,
                                                 int tid, int nthreads) {
    for (int idx = tid; idx < G * kD; idx += nthreads) {
        const int hh = idx / kD, dd = idx % kD;
        if (n_i <= 1) {
            const int64_t o = (int64_t)row * p.Hq + kvh * G + hh;
            p.out[o * kD + dd] = __float2half_rn(0.f);
            if (p.lse && dd == 0) p.lse[o] = -INFINITY;
        } else {
            p.part_acc[(slot * G + hh) * kD + dd] = 0.f;
            if (dd == 0) {
                p.part_m[slot * G + hh] = -INFINITY;
                p.part_l[slot * G + hh] = 0.f;
            }
        }
    }
}

// Combines the NW warp states in `cb` and stores the task's result: direct FP16 output when the
// row has one split, else the FP32 partial state in its compact slot;
// in FUSED mode the CTA that completes the last split of (row, kvh) merges in place
// (PAPER.md:77).  Called by `nthreads` threads (tid 0..nthreads-1) that synchronise on named
// barrier `bar_id`; the caller has already synchronised after filling `cb`.
template <int G, int NW>
__device__ __forceinline__ void finalize_task(const DecodeParams& p, CombineBuf<G, NW>& cb, int row, int kvh,
                                              int split, int n_i, int64_t slot, int tid, int nthreads,
                                              int bar_id) {
    for (int idx = tid; idx < G * kD; idx += nthreads) {
        const int hh = idx / kD, dd = idx % kD;
        float M = -INFINITY;
#pragma unroll
        for (int w = 0; w < NW; ++w) M = fmaxf(M, cb.m[w][hh]);
        float L = 0.f, A = 0.f;
#pragma unroll
        for (int w = 0; w < NW; ++w) {
            const float wgt = ex2_approx((cb.m[w][hh] - M) * p.scale_log2);  // m = -inf -> 0
            L += wgt * cb.l[w][hh];
            A += wgt * cb.acc[w][hh][dd];
        }
        if (n_i <= 1) {
            const int64_t o = (int64_t)row * p.Hq + kvh * G + hh;
            p.out[o * kD + dd] = __float2half_rn(A / L);
            if (p.lse && dd == 0) p.lse[o] = M * p.scale + logf(L);
        } else {
            p.part_acc[(slot * G + hh) * kD + dd] = A;
            if (dd == 0) {
                p.part_m[slot * G + hh] = M * p.scale;
                p.part_l[slot * G + hh] = L;
            }
        }
    }
    if (n_i > 1 && p.merge_mode == PKV_MERGE_FUSED) {
        __threadfence();  // partial state visible device-wide before the completion count
        named_bar_sync(bar_id, nthreads);
        if (tid == 0) {
            const int old = atomicAdd(&p.fuse_counters[row * p.Hkv + kvh], 1);
            const int last = (old == n_i - 1);
            if (last) p.fuse_counters[row * p.Hkv + kvh] = 0;  // self-reset for the next replay
            cb.flag = last;
        }
        named_bar_sync(bar_id, nthreads);
        if (cb.flag) {
            __threadfence();
            const int64_t base = slot - split;  // first slot of (row, kvh): DESIGN.md A8
            for (int idx = tid; idx < G * kD; idx += nthreads) merge_one<G>(p, base, n_i, row, kvh, idx / kD, idx % kD);
        }
    }
    named_bar_sync(bar_id, nthreads);  // cb may be refilled after this
}

// Rows with N_i = 0 emit no task in the workqueue route: out = 0, lse = -inf (A9).
__device__ __forceinline__ void zero_empty_rows(const DecodeParams& p) {
    const int per_row = p.Hq * kD;
    for (int i = blockIdx.x; i < p.B; i += gridDim.x) {
        if (p.seq_lens[i] > 0) continue;
        for (int e = threadIdx.x; e < per_row; e += blockDim.x) {
            p.out[(int64_t)i * per_row + e] = __float2half_rn(0.f);
            if (p.lse && e < p.Hq) p.lse[(int64_t)i * p.Hq + e] = -INFINITY;
        }
    }
}

// launchers implemented in the .cu files
cudaError_t launch_decode_simt(const DecodeParams& p, int G, int grid, cudaStream_t stream);
cudaError_t launch_decode_tma(const DecodeParams& p, int G, int grid, const void* tmap_k, const void* tmap_v,
                              cudaStream_t stream);
cudaError_t launch_builder(const pkv_shape& shape, const Resolved& rp, const int32_t* seq_lens_dev,
                           QueueHeader* hdr, int32_t* split_offsets, int32_t* fuse_counters, pkv_task* tasks,
                           int64_t tasks_cap, cudaStream_t stream);
cudaError_t launch_merge(const DecodeParams& p, int G, cudaStream_t stream);
int decode_tma_smem_bytes(int G);

}  // namespace pkv
