// pkv_decode_simt.cu -- PKV_KERNEL_SIMT: the plain-ALU decode kernel.
//
// One CTA (4 warps) per task, persistent grid-stride loop over the task list.  Each half-warp
// owns one token at a time: 16 lanes x 16-byte vector loads cover the 256-byte K (then V) row of
// the task's KV head, read straight from global memory through the block table (PAPER.md:50 page
// accessor).  The G query heads of the group share the loaded row: G dot products
// reduced with warp shuffles, exact online softmax (m, l, acc) in FP32.
// This is the kernel the SURVEY's issue-slot estimate is about (about 40 issue slots per 512 B):
// it is kept as the measured baseline that justifies the tensor-core tile loop of
// pkv_decode_tma.cu, and as an independent second implementation for parity tests.
#include "pkv_device.cuh"

namespace pkv {

namespace {

constexpr int kWarps = 4;
constexpr int kThreads = kWarps * 32;
constexpr int kUnroll = 4;  // tokens in flight per half-warp

__device__ __forceinline__ uint4 ldg_nc_16(const void* ptr) {
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
                 : "l"(ptr));
    return r;
}

__device__ __forceinline__ void unpack8(const uint4& u, float (&f)[8]) {
    const __half2* h = reinterpret_cast<const __half2*>(&u);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const float2 t = __half22float2(h[i]);
        f[2 * i] = t.x;
        f[2 * i + 1] = t.y;
    }
}

template <int G>
__global__ void __launch_bounds__(kThreads) pkv_decode_simt_kernel(const DecodeParams p) {
    __shared__ CombineBuf<G, kWarps> cb;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int hw = lane >> 4;   // half-warp: which of the warp's two tokens
    const int ch = lane & 15;   // 16-byte chunk of the 256-byte row: channels ch*8 .. ch*8+7

    pdl_launch_dependents();
    pdl_wait();
    zero_empty_rows(p);
    if (blockIdx.x == 0 && tid == 0) {   // this launch's mark (pkv_counters.launched_*)
        p.hdr->launched_decode = 1;
        p.hdr->launched_merge = 0;
    }
    const int num_tasks = p.hdr->num_tasks;
    for (int t = blockIdx.x; t < num_tasks; t += gridDim.x) {
        const pkv_task task = p.tasks[t];
        const int row = task.row, kvh = task.kvh;
        const int orow = request_row(p.row_index, row);   // row of q, out, lse, block_table, seq_lens
        const int N = plan_len(p.plan, p.seq_lens[orow]);
        const int so = p.split_offsets[row];
        const int n_i = p.split_offsets[row + 1] - so;
        const int64_t slot = (int64_t)so * p.Hkv + (int64_t)kvh * n_i + task.split;
        const int tok0 = task.t_begin * p.tile_tokens;
        const int tok1 = min(task.t_end * p.tile_tokens, N);
        if (tok0 >= tok1) {  // empty split: neutral state, before loading Q
            store_empty_task<G, kWarps>(p, &cb.flag[0], row, orow, kvh, task.split, n_i, slot, tid, 0);
            continue;
        }

        float qf[G][8];
#pragma unroll
        for (int g = 0; g < G; ++g) {
            const uint4 u = *reinterpret_cast<const uint4*>(p.q + ((int64_t)orow * p.Hq + kvh * G + g) * kD + ch * 8);
            unpack8(u, qf[g]);
        }
        float m[G], l[G], acc[G][8];
#pragma unroll
        for (int g = 0; g < G; ++g) {
            m[g] = -INFINITY;
            l[g] = 0.f;
#pragma unroll
            for (int c = 0; c < 8; ++c) acc[g][c] = 0.f;
        }

        const int32_t* bt = p.block_table + (int64_t)orow * p.max_pages;
        const int64_t head_off = (int64_t)kvh * p.stride_head + ch * 8;
        // the CTA walks 8 tokens per step (4 warps x 2 half-warps); kUnroll steps are in flight
        for (int base = tok0 + warp * 2; base < tok1; base += 8 * kUnroll) {  // warp-uniform bound
            uint4 ku[kUnroll], vu[kUnroll];
#pragma unroll
            for (int u = 0; u < kUnroll; ++u) {
                const int j = base + hw + 8 * u;
                if (j < tok1) {
                    const int64_t page = checked_page(bt[j >> (4 + p.page_shift)], p.plan.flags, p.num_pages, &p.hdr->error_word);
                    const int64_t off = page * p.stride_page + (int64_t)(j & ((16 << p.page_shift) - 1)) * p.stride_token + head_off;
                    ku[u] = ldg_nc_16(p.k_cache + off);
                    vu[u] = ldg_nc_16(p.v_cache + off);
                } else {
                    ku[u] = make_uint4(0, 0, 0, 0);
                    vu[u] = make_uint4(0, 0, 0, 0);
                }
            }
#pragma unroll
            for (int u = 0; u < kUnroll; ++u) {
                const int j = base + hw + 8 * u;
                const bool valid = j < tok1;  // uniform within the half-warp
                float kf[8], vf[8];
                unpack8(ku[u], kf);
                unpack8(vu[u], vf);
                float s[G];
#pragma unroll
                for (int g = 0; g < G; ++g) {
                    float d = 0.f;
#pragma unroll
                    for (int c = 0; c < 8; ++c) d = fmaf(qf[g][c], kf[c], d);
                    s[g] = d;
                }
#pragma unroll
                for (int off = 8; off >= 1; off >>= 1) {
#pragma unroll
                    for (int g = 0; g < G; ++g) s[g] += __shfl_xor_sync(0xffffffffu, s[g], off);
                }
                if (valid) {
#pragma unroll
                    for (int g = 0; g < G; ++g) {
                        const float mn = fmaxf(m[g], s[g]);
                        const float alpha = ex2_approx((m[g] - mn) * p.scale_log2);  // m = -inf -> 0
                        const float pw = ex2_approx((s[g] - mn) * p.scale_log2);
                        m[g] = mn;
                        l[g] = l[g] * alpha + pw;
#pragma unroll
                        for (int c = 0; c < 8; ++c) acc[g][c] = fmaf(acc[g][c], alpha, pw * vf[c]);
                    }
                }
            }
        }

        // the two half-warps of a warp hold states of disjoint token sets: combine in registers
#pragma unroll
        for (int g = 0; g < G; ++g) {
            const float mo = __shfl_xor_sync(0xffffffffu, m[g], 16);
            const float lo = __shfl_xor_sync(0xffffffffu, l[g], 16);
            const float mn = fmaxf(m[g], mo);
            const float a_self = (m[g] == -INFINITY) ? 0.f : ex2_approx((m[g] - mn) * p.scale_log2);
            const float a_oth = (mo == -INFINITY) ? 0.f : ex2_approx((mo - mn) * p.scale_log2);
            l[g] = l[g] * a_self + lo * a_oth;
#pragma unroll
            for (int c = 0; c < 8; ++c) {
                const float ao = __shfl_xor_sync(0xffffffffu, acc[g][c], 16);
                acc[g][c] = acc[g][c] * a_self + ao * a_oth;
            }
            m[g] = mn;
        }
        if (hw == 0) {
#pragma unroll
            for (int g = 0; g < G; ++g) {
#pragma unroll
                for (int c = 0; c < 8; ++c) cb.acc[warp][g][ch * 8 + c] = acc[g][c];
                if (ch == 0) {
                    cb.m[warp][g] = m[g];
                    cb.l[warp][g] = l[g];
                }
            }
        }
        __syncthreads();
        finalize_task<G, kWarps, kWarps>(p, cb, 0, 1, row, orow, kvh, task.split, n_i, slot, tid, 0, 0, p.scale, p.scale_log2);
    }
}

}  // namespace

cudaError_t launch_decode_simt(const DecodeParams& p, int G, int grid, cudaStream_t stream) {
    if (grid <= 0) return cudaSuccess;
    const bool pdl = !(p.plan.flags & PKV_FLAG_NO_PDL);
    if (G == 1) return launch_pdl(pdl, pkv_decode_simt_kernel<1>, dim3(grid), dim3(kThreads), 0, stream, p);
    if (G == 2) return launch_pdl(pdl, pkv_decode_simt_kernel<2>, dim3(grid), dim3(kThreads), 0, stream, p);
    if (G == 4) return launch_pdl(pdl, pkv_decode_simt_kernel<4>, dim3(grid), dim3(kThreads), 0, stream, p);
    if (G == 16) return launch_pdl(pdl, pkv_decode_simt_kernel<16>, dim3(grid), dim3(kThreads), 0, stream, p);
    return launch_pdl(pdl, pkv_decode_simt_kernel<8>, dim3(grid), dim3(kThreads), 0, stream, p);
}

}  // namespace pkv
