// pkv_api.cu -- the CUDA-facing entry points of include/pkv.h: argument checks, tensor-map
// encoding, workspace carving and the launch sequence [builder] -> decode -> [merge].
// No allocation, no synchronisation and no host read of device data in pkv_build_workqueue,
// pkv_decode and pkv_merge (they are CUDA-graph-capture-safe).
#include <cuda.h>

#include <cmath>
#include <cstring>
#include <vector>

#include "pkv_device.cuh"

namespace pkv {

namespace {

#ifdef PKV_TRACE
unsigned long long* g_trace = nullptr;  // trace build only (pkv_debug_set_trace)
#endif

int device_sm_count() {
    thread_local int cache[64];
    thread_local bool have[64] = {};
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return 0;
    if (!have[dev]) {
        int n = 0;
        if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return 0;
        cache[dev] = n;
        have[dev] = true;
    }
    return cache[dev];
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn() {
    static EncodeTiledFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        void* ptr = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ptr, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(ptr);
        tried = true;
    }
    return fn;
}

typedef CUresult (*MemsetD32Fn)(CUdeviceptr, unsigned int, size_t, CUstream);
MemsetD32Fn memset_d32_fn() {
    static MemsetD32Fn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        void* ptr = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuMemsetD32Async", &ptr, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<MemsetD32Fn>(ptr);
        tried = true;
    }
    return fn;
}

struct Strides { int64_t page, token, head; };
Strides effective_strides(const pkv_shape& s) {
    if (s.kv_stride_page == 0) return {(int64_t)s.page_size * s.Hkv * s.d, (int64_t)s.Hkv * s.d, (int64_t)s.d};
    return {s.kv_stride_page, s.kv_stride_token, s.kv_stride_head};
}

// Rank-5 tensor map over one cache: dims (64 ch, P tok, 2 ch-halves, Hkv heads, pages), strides
// from the caller's layout, box (64, 16, 2, HG, 1): the HG-head slice of one 16-token block of a
// page (the whole page when P = 16), landing in
// shared memory as [head][ch-half][tok][64 ch] with the 128-byte swizzle (conflict-free ldmatrix).
bool encode_map(const void* base, const pkv_shape& s, const Strides& st, int HG, CUtensorMap* out) {
    EncodeTiledFn fn = encode_fn();
    if (!fn) return false;
    const cuuint64_t pages = (cuuint64_t)(s.num_pages > 0 ? s.num_pages : 1);
    const bool fp8 = s.kv_dtype != PKV_KV_F16;           // one-byte caches (E4M3, INT8)
    const cuuint64_t eb = fp8 ? 1 : 2;                   // bytes per element
    const cuuint32_t inner = (cuuint32_t)(128 / eb);     // elements of one 128-byte swizzled row
    const cuuint32_t blocks = (cuuint32_t)(s.d / inner); // 128-byte blocks of a head's row
    cuuint64_t dims[5] = {inner, (cuuint64_t)s.page_size, blocks, (cuuint64_t)s.Hkv, pages};
    cuuint64_t strides[4] = {(cuuint64_t)st.token * eb, 128, (cuuint64_t)st.head * eb, (cuuint64_t)st.page * eb};
    cuuint32_t box[5] = {inner, 16, blocks, (cuuint32_t)HG, 1};
    cuuint32_t estr[5] = {1, 1, 1, 1, 1};
    const CUresult r = fn(out, fp8 ? CU_TENSOR_MAP_DATA_TYPE_UINT8 : CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 5, const_cast<void*>(base), dims, strides, box, estr,
                          CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                          CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS;
}

struct MapCacheEntry {
    const void* base;
    int64_t num_pages, sp, st, sh;
    int32_t Hkv, HG, P, d, dt;
    CUtensorMap map;
};

// Returns the tensor map of `base` for HG heads per box, encoding it on first use (per thread).
const CUtensorMap* get_map(const void* base, const pkv_shape& s, int HG) {
    constexpr int kCap = 32;
    thread_local MapCacheEntry cache[kCap];   // fixed storage: returned pointers stay valid
    thread_local int count = 0, next = 0;
    const Strides st = effective_strides(s);
    for (int i = 0; i < count; ++i) {
        const MapCacheEntry& e = cache[i];
        if (e.base == base && e.num_pages == s.num_pages && e.sp == st.page && e.st == st.token && e.sh == st.head &&
            e.Hkv == s.Hkv && e.HG == HG && e.P == s.page_size && e.d == s.d && e.dt == s.kv_dtype)
            return &e.map;
    }
    MapCacheEntry e;
    e.base = base; e.num_pages = s.num_pages; e.sp = st.page; e.st = st.token; e.sh = st.head; e.Hkv = s.Hkv; e.HG = HG; e.P = s.page_size; e.d = s.d; e.dt = s.kv_dtype;
    if (!encode_map(base, s, st, HG, &e.map)) return nullptr;
    const int slot = count < kCap ? count++ : (next = (next + 1) % kCap);
    cache[slot] = e;
    return &cache[slot].map;
}

pkv_status cuda_fail(cudaError_t e, const char* what) {
    set_error("%s: %s", what, cudaGetErrorString(e));
    return PKV_ERR_CUDA;
}

struct QueuePtrs {
    QueueHeader* hdr;
    int32_t* split_offsets;
    RowSlot* rowslots;
    pkv_task* tasks;
};

struct WsPtrs {
    QueuePtrs q;
    int32_t* fuse_counters;
    float *part_m, *part_l, *part_acc;
};

WsPtrs carve(void* workspace, const WorkspaceLayout& L) {
    unsigned char* w = static_cast<unsigned char*>(workspace);
    WsPtrs r;
    r.q.hdr = reinterpret_cast<QueueHeader*>(w + L.header);
    r.q.split_offsets = reinterpret_cast<int32_t*>(w + L.split_offsets);
    r.q.rowslots = reinterpret_cast<RowSlot*>(w + L.rowslots);
    r.q.tasks = reinterpret_cast<pkv_task*>(w + L.tasks);
    r.fuse_counters = reinterpret_cast<int32_t*>(w + L.fuse_counters);
    r.part_m = reinterpret_cast<float*>(w + L.part_m);
    r.part_l = reinterpret_cast<float*>(w + L.part_l);
    r.part_acc = reinterpret_cast<float*>(w + L.part_acc);
    return r;
}

pkv_status check_workspace(const void* workspace, size_t bytes, const WorkspaceLayout& L) {
    if (!workspace) { set_error("null workspace"); return PKV_ERR_INVALID_ARG; }
    if (reinterpret_cast<uintptr_t>(workspace) % 256) { set_error("workspace must be 256-byte aligned"); return PKV_ERR_INVALID_ARG; }
    if (bytes < L.total) { set_error("workspace has %zu bytes, %zu needed", bytes, L.total); return PKV_ERR_WORKSPACE; }
    return PKV_OK;
}

// Launches decode (+ merge).  known_tasks / known_max_n >= 0: the queue was planned on the host,
// so launches that have nothing to do are skipped (A13).
pkv_status run_decode(const pkv_shape& s, const Resolved& rp, const void* q, const void* k_cache, const void* v_cache,
                      const int32_t* block_table, const int32_t* seq_lens, const int32_t* row_index, void* out, float* lse, float scale,
                      const pkv_append* append,
                      const QueuePtrs& qp, const WsPtrs& ws, int64_t known_tasks, int known_max_n, int64_t known_slots,
                      int num_sms, uint32_t stages, bool fused_build, int64_t tasks_cap,
                      cudaStream_t stream, int* decode_launches, int* merge_launches) {
    DecodeParams p;
    std::memset(&p, 0, sizeof(p));
    const Strides st = effective_strides(s);
    p.q = static_cast<const __half*>(q);
    p.k_cache = static_cast<const __half*>(k_cache);
    p.v_cache = static_cast<const __half*>(v_cache);
    p.block_table = block_table;
    p.seq_lens = seq_lens;
    p.row_index = row_index;
    p.tasks = qp.tasks;
    p.rowslots = qp.rowslots;
    p.split_offsets = qp.split_offsets;
    p.hdr = qp.hdr;
    p.out = static_cast<__half*>(out);
    p.lse = lse;
    p.part_m = ws.part_m; p.part_l = ws.part_l; p.part_acc = ws.part_acc;
    p.fuse_counters = ws.fuse_counters;
    p.stride_page = st.page; p.stride_token = st.token; p.stride_head = st.head;
    p.B = s.B; p.Hq = s.Hq; p.Hkv = s.Hkv; p.max_pages = s.max_pages; p.d = s.d;
    p.k_scale = s.k_scale; p.v_scale = s.v_scale;
    if (append) {
        p.k_new = static_cast<const __half*>(append->k_new);
        p.v_new = static_cast<const __half*>(append->v_new);
        p.rope_cos = append->rope_cos;
        p.rope_sin = append->rope_sin;
        p.rope_positions = append->rope_positions;
    }
    p.tile_tokens = rp.tile_tokens; p.merge_mode = rp.merge_mode;
    p.dynamic_sched = 1;
    p.force_replan = (rp.flags & PKV_FLAG_TEST_REPLAN) ? 1 : 0;
    p.plan = make_plan_args(s, rp);
    p.plan.row_index = row_index;
    p.tasks_cap = tasks_cap;
    p.fused_build = fused_build ? 1 : 0;
    p.num_pages = s.num_pages;
    p.page_shift = s.page_size == 64 ? 2 : (s.page_size == 32 ? 1 : 0);
#ifdef PKV_TRACE
    p.trace = g_trace;
#endif
    const float sc = scale > 0.f ? scale : 1.0f / std::sqrt((float)s.d);
    p.scale = sc;
    p.scale_log2 = sc * kLog2e;

    if (decode_launches) *decode_launches = 0;
    if (merge_launches) *merge_launches = 0;
    if (s.B == 0) return PKV_OK;
    const int64_t bound = known_tasks >= 0 ? known_tasks : (int64_t)s.B * s.Hkv * rp.S;
    cudaError_t e;
    if (known_tasks == 0 && (stages & PKV_STAGE_DECODE)) {
        // every row is empty: out = 0, lse = -inf, no decode launch
        e = cudaMemsetAsync(out, 0, (size_t)s.B * s.Hq * s.d * 2, stream);
        if (e != cudaSuccess) return cuda_fail(e, "memset out");
        if (lse) {
            MemsetD32Fn ms = memset_d32_fn();
            if (!ms || ms(reinterpret_cast<CUdeviceptr>(lse), 0xff800000u /* -inf */, (size_t)s.B * s.Hq, stream) !=
                           CUDA_SUCCESS) {
                set_error("cuMemsetD32Async failed");
                return PKV_ERR_CUDA;
            }
        }
    }
    if (known_tasks != 0 && (stages & PKV_STAGE_DECODE)) {
        if (rp.kernel == PKV_KERNEL_TMA_MMA) {
            // (row, split) pairs the queue will hold: known when planned on the host, else a bound.
            // BALANCED aims at a single wave of at most U = policy.num_sms pairs, so a caller that
            // passes U = SMs * HG / Hkv gets HG heads per CTA and one unit per SM.
            int64_t row_slots = known_slots >= 0 ? known_slots : (int64_t)s.B * rp.S;
            if (known_slots < 0 && rp.split_mode == PKV_SPLIT_BALANCED && rp.num_sms > 0 && rp.num_sms < row_slots)
                row_slots = rp.num_sms;
            const int HG = choose_heads_per_cta(rp.heads_per_cta, s.Hkv, row_slots, num_sms, max_heads_per_cta(rp.G, s.d));
            p.prefetch_pages = rp.prefetch_kb * 1024 / decode_tma_stage_bytes(HG, s.d, s.kv_dtype != PKV_KV_F16);
            // by value: inserting the V map may evict the cache entry the K pointer refers to
            const CUtensorMap* pk = get_map(k_cache, s, HG);
            CUtensorMap mk_copy, mv_copy;
            if (pk) mk_copy = *pk;
            const CUtensorMap* pv = get_map(v_cache, s, HG);
            if (pv) mv_copy = *pv;
            if (!pk || !pv) {
                set_error("cuTensorMapEncodeTiled failed for the K/V cache (base %p/%p)", k_cache, v_cache);
                return PKV_ERR_CUDA;
            }
            const CUtensorMap *mk = &mk_copy, *mv = &mv_copy;
            p.heads_per_cta = HG;
            // Units are handed out by an atomic counter only when every head has ONE compute warp
            // (HG = 8): with several warps per head the page-to-warp assignment follows the CTA's
            // stream position, so a dynamic hand-out would make the FP32 combine order -- and the
            // last bits of the result -- depend on which units a CTA drew before.  Round-robin
            // keeps every launch bitwise reproducible.
            p.dynamic_sched = HG * (rp.G == 16 ? 2 : 1) == 8 ? 1 : 0;
            const int64_t units = row_slots * (s.Hkv / HG);
            const int grid = (int)(units < num_sms ? units : num_sms);
            e = launch_decode_tma(p, rp.G, HG, s.d, s.kv_dtype, grid, mk, mv, stream);
        } else {
            const int64_t cap = (int64_t)num_sms * 4;
            const int grid = (int)(bound < cap ? bound : cap);
            e = launch_decode_simt(p, rp.G, grid, stream);
        }
        if (e != cudaSuccess) return cuda_fail(e, "decode launch");
        if (decode_launches) *decode_launches = 1;
    }
    const bool need_merge = (stages & PKV_STAGE_MERGE) && rp.merge_mode == PKV_MERGE_SEPARATE &&
                            (known_max_n >= 0 ? known_max_n > 1 : rp.S > 1) && known_tasks != 0;
    if (need_merge) {
        e = launch_merge(p, rp.G, stream);
        if (e != cudaSuccess) return cuda_fail(e, "merge launch");
        if (merge_launches) *merge_launches = 1;
    }
    return PKV_OK;
}

pkv_status check_decode_ptrs(const pkv_shape& s, const void* q, const void* k, const void* v, const int32_t* bt,
                             const int32_t* sl, const void* out) {
    if (s.B > 0 && (!q || !k || !v || !bt || !sl || !out)) { set_error("null pointer argument"); return PKV_ERR_INVALID_ARG; }
    if ((reinterpret_cast<uintptr_t>(q) | reinterpret_cast<uintptr_t>(k) | reinterpret_cast<uintptr_t>(v) |
         reinterpret_cast<uintptr_t>(out)) % 16) {
        set_error("q, k_cache, v_cache and out must be 16-byte aligned");
        return PKV_ERR_INVALID_ARG;
    }
    return PKV_OK;
}

}  // namespace
}  // namespace pkv

using namespace pkv;

extern "C" {

#ifdef PKV_TRACE
// Trace build only (python -m paper_2606_26666_b200.build --trace): device buffer of grid*16
// uint64 that the TMA decode kernel fills with %globaltimer stamps of its phases; NULL = off.
__attribute__((visibility("default"))) void pkv_debug_set_trace(void* dev) { g_trace = static_cast<unsigned long long*>(dev); }
#endif

pkv_status pkv_build_workqueue(const pkv_shape* shape, const pkv_split_policy* policy, const int32_t* seq_lens_dev,
                               void* workspace, size_t workspace_bytes, void* stream) {
    clear_error();
    Resolved rp;
    pkv_status st = validate_and_resolve(shape, policy, device_sm_count(), false, &rp);
    if (st != PKV_OK) return st;
    if (!seq_lens_dev && shape->B > 0) { set_error("null seq_lens"); return PKV_ERR_INVALID_ARG; }
    const WorkspaceLayout L = workspace_layout(*shape, rp.S);
    st = check_workspace(workspace, workspace_bytes, L);
    if (st != PKV_OK) return st;
    const WsPtrs ws = carve(workspace, L);
    const cudaError_t e = launch_builder(*shape, rp, seq_lens_dev, nullptr, ws.q.hdr, ws.q.split_offsets, ws.fuse_counters,
                                         ws.q.rowslots, ws.q.tasks, L.slots_cap, static_cast<cudaStream_t>(stream));
    if (e != cudaSuccess) return cuda_fail(e, "builder launch");
    return PKV_OK;
}

}  // extern "C"

namespace {

pkv_status decode_stages(const pkv_shape* shape, const pkv_split_policy* policy, const void* q,
                             const void* k_cache, const void* v_cache, const int32_t* block_table,
                             const int32_t* seq_lens, const int32_t* row_index, void* out, float* lse, float scale,
                             uint32_t stages, void* workspace, size_t workspace_bytes, void* stream,
                             const pkv_shape* layout_shape = nullptr, const pkv_append* append = nullptr) {
    // layout_shape: the shape the workspace is carved for (pkv_decode_buckets: the whole batch, so
    // that the header and the completion counters sit at the same place for every bucket)
    clear_error();
    Resolved rp;
    const int sms = device_sm_count();
    pkv_status st = validate_and_resolve(shape, policy, sms, false, &rp);
    if (st != PKV_OK) return st;
    if (sms <= 0) { set_error("no CUDA device"); return PKV_ERR_CUDA; }
    if (stages & ~(uint32_t)PKV_STAGE_ALL) { set_error("unknown stage bits 0x%x", stages); return PKV_ERR_INVALID_ARG; }
    st = check_decode_ptrs(*shape, q, k_cache, v_cache, block_table, seq_lens, out);
    if (st != PKV_OK) return st;
    const WorkspaceLayout L = workspace_layout(layout_shape ? *layout_shape : *shape, rp.S);
    st = check_workspace(workspace, workspace_bytes, L);
    if (st != PKV_OK) return st;
    const WsPtrs ws = carve(workspace, L);
    cudaStream_t cs = static_cast<cudaStream_t>(stream);
    // The TMA kernel derives the queue itself (fused build) when it runs in the same call;
    // otherwise (builder alone, SIMT kernel, very large batches) the builder kernel runs first.
    const bool fused = (stages & PKV_STAGE_BUILD) && (stages & PKV_STAGE_DECODE) && !(rp.flags & PKV_FLAG_SEPARATE_BUILD) &&
                       rp.kernel == PKV_KERNEL_TMA_MMA && shape->B <= kMaxFusedRows;
    if ((stages & PKV_STAGE_BUILD) && !fused) {
        const cudaError_t e = launch_builder(*shape, rp, seq_lens, row_index, ws.q.hdr, ws.q.split_offsets, ws.fuse_counters,
                                             ws.q.rowslots, ws.q.tasks, L.slots_cap, cs);
        if (e != cudaSuccess) return cuda_fail(e, "builder launch");
    }
    if (append) {
        if (!append->k_new || !append->v_new || (append->rope_cos == nullptr) != (append->rope_sin == nullptr) ||
            (append->rope_cos && append->rope_positions <= 0)) {
            set_error("pkv_decode_append: k_new / v_new null, or only one RoPE table, or rope_positions <= 0");
            return PKV_ERR_INVALID_ARG;
        }
        if (rp.kernel != PKV_KERNEL_TMA_MMA || shape->d != kD) {
            set_error("pkv_decode_append needs the TMA kernel and d = 128");
            return PKV_ERR_UNSUPPORTED;
        }
    }
    return run_decode(*shape, rp, q, k_cache, v_cache, block_table, seq_lens, row_index, out, lse, scale, append, ws.q, ws, -1, -1,
                      -1, sms, stages, fused, L.slots_cap, cs, nullptr, nullptr);
}

}  // namespace

extern "C" {

pkv_status pkv_decode_stages(const pkv_shape* shape, const pkv_split_policy* policy, const void* q,
                             const void* k_cache, const void* v_cache, const int32_t* block_table,
                             const int32_t* seq_lens, void* out, float* lse, float scale, uint32_t stages,
                             void* workspace, size_t workspace_bytes, void* stream) {
    return decode_stages(shape, policy, q, k_cache, v_cache, block_table, seq_lens, nullptr, out, lse, scale, stages,
                         workspace, workspace_bytes, stream);
}

pkv_status pkv_decode_indexed(const pkv_shape* shape, const pkv_split_policy* policy, const void* q,
                              const void* k_cache, const void* v_cache, const int32_t* block_table,
                              const int32_t* seq_lens, const int32_t* row_index, void* out, float* lse, float scale,
                              void* workspace, size_t workspace_bytes, void* stream) {
    if (shape && shape->B > kMaxFusedRows) {
        clear_error();
        set_error("pkv_decode_indexed: at most %d indexed rows per launch", kMaxFusedRows);
        return PKV_ERR_UNSUPPORTED;
    }
    if (shape && shape->B > 0 && !row_index) {
        clear_error();
        set_error("null row_index");
        return PKV_ERR_INVALID_ARG;
    }
    return decode_stages(shape, policy, q, k_cache, v_cache, block_table, seq_lens, row_index, out, lse, scale,
                         PKV_STAGE_ALL, workspace, workspace_bytes, stream);
}

pkv_status pkv_decode_append(const pkv_shape* shape, const pkv_split_policy* policy, const void* q, void* k_cache,
                             void* v_cache, const int32_t* block_table, const int32_t* seq_lens, const int32_t* row_index,
                             const pkv_append* append, void* out, float* lse, float scale, void* workspace,
                             size_t workspace_bytes, void* stream) {
    if (!append) {
        clear_error();
        set_error("pkv_decode_append: null append");
        return PKV_ERR_INVALID_ARG;
    }
    if (row_index && shape && shape->B > kMaxFusedRows) {
        clear_error();
        set_error("pkv_decode_append: at most %d indexed rows per launch", kMaxFusedRows);
        return PKV_ERR_UNSUPPORTED;
    }
    return decode_stages(shape, policy, q, k_cache, v_cache, block_table, seq_lens, row_index, out, lse, scale, PKV_STAGE_ALL,
                         workspace, workspace_bytes, stream, nullptr, append);
}

pkv_status pkv_decode_buckets(const pkv_shape* shape, const pkv_split_policy* policy, const void* q,
                              const void* k_cache, const void* v_cache, const int32_t* block_table,
                              const int32_t* seq_lens, const int32_t* row_index, const int32_t* bucket_offsets_host,
                              int32_t num_buckets, void* out, float* lse, float scale, void* workspace,
                              size_t workspace_bytes, void* stream) {
    clear_error();
    if (!shape || !policy || num_buckets < 0 || (num_buckets > 0 && (!bucket_offsets_host || !row_index))) {
        set_error("pkv_decode_buckets: null argument");
        return PKV_ERR_INVALID_ARG;
    }
    if (bucket_offsets_host && (bucket_offsets_host[0] != 0 || bucket_offsets_host[num_buckets] > shape->B)) {
        set_error("pkv_decode_buckets: bucket_offsets must start at 0 and end at or below B");
        return PKV_ERR_INVALID_ARG;
    }
    // every bucket is a launch pair of its own over the bucket's rows ("one per route
    // length"); then one more indexed launch for the rows that belong to no bucket (N_i = 0: out = 0)
    const int32_t nb_rows = num_buckets > 0 ? bucket_offsets_host[num_buckets] : 0;
    for (int32_t b = 0; b <= num_buckets; ++b) {
        const int32_t lo = b < num_buckets ? bucket_offsets_host[b] : nb_rows;
        const int32_t hi = b < num_buckets ? bucket_offsets_host[b + 1] : shape->B;
        if (hi < lo) { set_error("pkv_decode_buckets: bucket_offsets must be non-decreasing"); return PKV_ERR_INVALID_ARG; }
        if (hi == lo) continue;
        pkv_shape sub = *shape;
        sub.B = hi - lo;
        if (sub.B > kMaxFusedRows) { set_error("pkv_decode_buckets: at most %d rows per bucket", kMaxFusedRows); return PKV_ERR_UNSUPPORTED; }
        const pkv_status st = decode_stages(&sub, policy, q, k_cache, v_cache, block_table, seq_lens, row_index + lo, out, lse,
                                            scale, PKV_STAGE_ALL, workspace, workspace_bytes, stream, shape);
        if (st != PKV_OK) return st;
    }
    return PKV_OK;
}

pkv_status pkv_decode(const pkv_shape* shape, const pkv_split_policy* policy, const void* q, const void* k_cache,
                      const void* v_cache, const int32_t* block_table, const int32_t* seq_lens, void* out, float* lse,
                      float scale, int32_t build_queue, void* workspace, size_t workspace_bytes, void* stream) {
    return pkv_decode_stages(shape, policy, q, k_cache, v_cache, block_table, seq_lens, out, lse, scale,
                             PKV_STAGE_DECODE | PKV_STAGE_MERGE | (build_queue ? PKV_STAGE_BUILD : 0), workspace,
                             workspace_bytes, stream);
}

pkv_status pkv_merge(const pkv_shape* shape, const float* part_m, const float* part_l, const float* part_acc,
                     const int32_t* split_offsets, void* out, float* lse, void* stream) {
    clear_error();
    pkv_split_policy pol;
    std::memset(&pol, 0, sizeof(pol));
    pol.tile_tokens = shape ? shape->page_size : 16;
    pol.num_splits = 1;
    Resolved rp;
    pkv_status st = validate_and_resolve(shape, &pol, 0, true, &rp);
    if (st != PKV_OK) return st;
    if (shape->B > 0 && (!part_m || !part_l || !part_acc || !split_offsets || !out)) {
        set_error("null pointer argument");
        return PKV_ERR_INVALID_ARG;
    }
    DecodeParams p;
    std::memset(&p, 0, sizeof(p));
    p.part_m = const_cast<float*>(part_m);
    p.part_l = const_cast<float*>(part_l);
    p.part_acc = const_cast<float*>(part_acc);
    p.split_offsets = const_cast<int32_t*>(split_offsets);
    p.hdr = nullptr;
    p.out = static_cast<__half*>(out);
    p.lse = lse;
    p.B = shape->B; p.Hq = shape->Hq; p.Hkv = shape->Hkv; p.d = shape->d;
    const cudaError_t e = launch_merge(p, rp.G, static_cast<cudaStream_t>(stream));
    if (e != cudaSuccess) return cuda_fail(e, "merge launch");
    return PKV_OK;
}

pkv_status pkv_get_counters(const pkv_shape* shape, const pkv_split_policy* policy, const void* workspace,
                            size_t workspace_bytes, pkv_counters* host_out, void* stream) {
    clear_error();
    Resolved rp;
    pkv_status st = validate_and_resolve(shape, policy, device_sm_count(), false, &rp);
    if (st != PKV_OK) return st;
    if (!host_out) { set_error("null host_out"); return PKV_ERR_INVALID_ARG; }
    const WorkspaceLayout L = workspace_layout(*shape, rp.S);
    st = check_workspace(workspace, workspace_bytes, L);
    if (st != PKV_OK) return st;
    QueueHeader h;
    cudaStream_t cs = static_cast<cudaStream_t>(stream);
    cudaError_t e = cudaMemcpyAsync(&h, static_cast<const unsigned char*>(workspace) + L.header, sizeof(h),
                                    cudaMemcpyDeviceToHost, cs);
    if (e == cudaSuccess) e = cudaStreamSynchronize(cs);
    if (e != cudaSuccess) return cuda_fail(e, "read header");
    std::memset(host_out, 0, sizeof(*host_out));
    host_out->tasks = h.num_tasks;
    host_out->empty_tasks = h.empty_tasks;
    host_out->decode_launches = h.num_tasks > 0 ? 1 : 0;
    host_out->merge_launches =
        (h.num_tasks > 0 && h.max_row_splits > 1 && rp.merge_mode == PKV_MERGE_SEPARATE) ? 1 : 0;
    host_out->build_launches = h.build_launches;
    host_out->useful_kv_bytes = h.sum_seq_lens * 2 * shape->Hkv * shape->d * (shape->kv_dtype != PKV_KV_F16 ? 1 : 2);
    host_out->merge_bytes = (int64_t)h.num_tasks * rp.G * (shape->d + 2) * 4;
    host_out->num_splits = h.resolved_splits;
    host_out->max_row_splits = h.max_row_splits;
    host_out->chunk_tiles = h.chunk_tiles;
    host_out->launched_build = h.launched_build;
    host_out->launched_decode = h.launched_decode;
    host_out->launched_merge = h.launched_merge;
    host_out->error_word = h.error_word;
    return PKV_OK;
}

pkv_status pkv_read_workqueue(const pkv_shape* shape, const pkv_split_policy* policy, const void* workspace,
                              size_t workspace_bytes, pkv_task* host_tasks, int32_t cap, int32_t* host_split_offsets,
                              int32_t* host_num_tasks, void* stream) {
    clear_error();
    Resolved rp;
    pkv_status st = validate_and_resolve(shape, policy, device_sm_count(), false, &rp);
    if (st != PKV_OK) return st;
    if (!host_num_tasks) { set_error("null host_num_tasks"); return PKV_ERR_INVALID_ARG; }
    const WorkspaceLayout L = workspace_layout(*shape, rp.S);
    st = check_workspace(workspace, workspace_bytes, L);
    if (st != PKV_OK) return st;
    const unsigned char* w = static_cast<const unsigned char*>(workspace);
    cudaStream_t cs = static_cast<cudaStream_t>(stream);
    QueueHeader h;
    cudaError_t e = cudaMemcpyAsync(&h, w + L.header, sizeof(h), cudaMemcpyDeviceToHost, cs);
    if (e == cudaSuccess) e = cudaStreamSynchronize(cs);
    if (e != cudaSuccess) return cuda_fail(e, "read header");
    *host_num_tasks = h.num_tasks;
    if (host_split_offsets) {
        e = cudaMemcpyAsync(host_split_offsets, w + L.split_offsets, sizeof(int32_t) * ((size_t)shape->B + 1),
                            cudaMemcpyDeviceToHost, cs);
        if (e != cudaSuccess) return cuda_fail(e, "read split_offsets");
    }
    if (host_tasks && cap > 0) {
        const int32_t n = h.num_tasks < cap ? h.num_tasks : cap;
        e = cudaMemcpyAsync(host_tasks, w + L.tasks, sizeof(pkv_task) * (size_t)n, cudaMemcpyDeviceToHost, cs);
        if (e != cudaSuccess) return cuda_fail(e, "read tasks");
    }
    e = cudaStreamSynchronize(cs);
    if (e != cudaSuccess) return cuda_fail(e, "sync");
    if (host_tasks && h.num_tasks > cap) { set_error("cap=%d < %d tasks", cap, h.num_tasks); return PKV_ERR_WORKSPACE; }
    return PKV_OK;
}

pkv_status pkv_workspace_partials(const pkv_shape* shape, const pkv_split_policy* policy, void* workspace,
                                  size_t workspace_bytes, float** part_m, float** part_l, float** part_acc,
                                  int64_t* slots_cap) {
    clear_error();
    Resolved rp;
    pkv_status st = validate_and_resolve(shape, policy, device_sm_count(), false, &rp);
    if (st != PKV_OK) return st;
    const WorkspaceLayout L = workspace_layout(*shape, rp.S);
    st = check_workspace(workspace, workspace_bytes, L);
    if (st != PKV_OK) return st;
    const WsPtrs ws = carve(workspace, L);
    if (part_m) *part_m = ws.part_m;
    if (part_l) *part_l = ws.part_l;
    if (part_acc) *part_acc = ws.part_acc;
    if (slots_cap) *slots_cap = L.slots_cap;
    return PKV_OK;
}

}  // extern "C"

// ------------------------------------------------------------------ host-buffer path

namespace pkv {
namespace {

// Image of one step's host inputs, identical in the pinned staging buffer and in dev_scratch:
//   [StageHeader][seq_lens B][q B*Hq*d f16][block_table B*max_pages]
// followed (device only) by the FP16 output.  seq_lens and q are adjacent: one H2D copy moves
// both.  The block table in `staging` is the SHADOW of what dev_scratch holds: a step uploads only
// the rows whose used entries differ from it (a growing row changes one entry every page_size steps).
struct StageHeader {
    uint64_t magic;
    const void* table_src;   // block_table_host the shadow was made from (informational)
    const void* dev;         // the dev_scratch the shadow mirrors
    int32_t B, max_pages;
    int64_t pad_[3];
};
constexpr uint64_t kStageMagic = 0x706b765f73746731ull;   // "pkv_stg1"

struct HostImage {
    size_t hdr, seq_lens, q, block_table, out, total;
};
HostImage host_image(const pkv_shape& s) {
    HostImage h;
    size_t off = 0;
    h.hdr = off;           off = align_up(off + sizeof(StageHeader), 256);
    h.seq_lens = off;      off = align_up(off + 4 * (size_t)s.B, 256);
    h.q = off;             off = align_up(off + 2 * (size_t)s.B * s.Hq * s.d, 256);
    h.block_table = off;   off = align_up(off + 4 * (size_t)s.B * s.max_pages, 256);
    h.out = off;           off = align_up(off + 2 * (size_t)s.B * s.Hq * s.d, 256);
    h.total = off;
    return h;
}

// Device pointer of a pinned, device-mapped host buffer (else nullptr).  use_cache (the caller set
// PKV_FLAG_OUT_PINNED: the buffer stays registered while the library sees it): the last answers are
// kept per thread, a serving loop passes the same few buffers every step and a pointer query costs
// about a microsecond.  Without it the driver is asked every time.
void* mapped_device_pointer(const void* host, size_t align, bool use_cache) {
    struct Entry { const void* host; void* dev; };
    thread_local Entry cache[8] = {};
    thread_local int next = 0;
    for (const Entry& e : cache)
        if (use_cache && e.host == host && host != nullptr && e.dev != nullptr)
            return reinterpret_cast<uintptr_t>(e.dev) % align == 0 ? e.dev : nullptr;
    cudaPointerAttributes attr;
    void* dev = nullptr;
    if (cudaPointerGetAttributes(&attr, host) == cudaSuccess && attr.type == cudaMemoryTypeHost && attr.devicePointer != nullptr)
        dev = attr.devicePointer;
    else
        (void)cudaGetLastError();   // an unregistered host pointer is not an error here
    if (use_cache && dev != nullptr) {
        cache[next] = Entry{host, dev};
        next = (next + 1) % 8;
    }
    return reinterpret_cast<uintptr_t>(dev) % align == 0 ? dev : nullptr;
}

// PKV_SPLIT_AUTO: the cost model's choice for these lengths.  The last choice is kept per thread and
// reused while the batch looks the same at a 128-token grain (a decode step adds one token per row:
// the estimate moves by parts in ten thousand, the argmin almost never).
pkv_status auto_policy(const pkv_shape& s, const pkv_split_policy& base, const int32_t* lens, int sms, pkv_split_policy* out) {
    struct Memo {
        std::vector<int32_t> coarse;
        pkv_split_policy base, chosen;
        int32_t Hq = 0, Hkv = 0, sms = 0;
        bool valid = false;
    };
    thread_local Memo memo;
    bool same = memo.valid && memo.Hq == s.Hq && memo.Hkv == s.Hkv && memo.sms == sms && (int32_t)memo.coarse.size() == s.B &&
                std::memcmp(&memo.base, &base, sizeof(base)) == 0;
    for (int32_t i = 0; same && i < s.B; ++i) same = memo.coarse[i] == (lens[i] > 0 ? (lens[i] >> 7) + 1 : 0);
    if (same) { *out = memo.chosen; return PKV_OK; }
    pkv_cost_model cm;
    pkv_default_cost_model(sms, &cm);
    const pkv_status st = pkv_choose_policy(&s, lens, &cm, &base, out, nullptr);
    if (st != PKV_OK) return st;
    memo.coarse.resize((size_t)s.B);
    for (int32_t i = 0; i < s.B; ++i) memo.coarse[i] = lens[i] > 0 ? (lens[i] >> 7) + 1 : 0;
    memo.base = base; memo.chosen = *out; memo.Hq = s.Hq; memo.Hkv = s.Hkv; memo.sms = sms; memo.valid = true;
    return PKV_OK;
}

// ------------------------------------------------------------------ pipelined host-buffer step
// (pkv_decode_host_pipelined).

// The pipeline's GPU-visible words, at byte 128 of the image header in the pinned, device-mapped
// staging buffer (word indices: pkv_device.cuh kPipe*Word).  flag: host -> GPU, the number of the last
// released step (the gate of step n waits for flag >= n).  GPU -> host: staged = the stage kernel of
// step n has finished reading the image; done = step n's result is in out_host; expired = step n's
// gate gave up waiting and the step ran on stale inputs.
struct PipeWords {
    uint32_t flag;
    uint32_t pad0_[15];
    uint32_t staged;
    uint32_t done;
    uint32_t expired;
    uint32_t pad1_[13];
};
static_assert(sizeof(StageHeader) <= 128 && sizeof(PipeWords) == 128, "image header: StageHeader | PipeWords in 256 bytes");
static_assert(offsetof(PipeWords, flag) == 4 * kPipeFlagWord && offsetof(PipeWords, staged) == 4 * kPipeStagedWord &&
              offsetof(PipeWords, done) == 4 * kPipeDoneWord && offsetof(PipeWords, expired) == 4 * kPipeExpiredWord, "PipeWords layout");
constexpr unsigned long long kGateTimeoutNs = 200ull * 1000 * 1000;   // an armed step nobody releases blocks the stream this long
constexpr size_t kPipeWordsOffset = 128;

// Host-only state of one pipeline (one per staging buffer, per thread).
struct PipeCtx {
    void* staging = nullptr;      // key
    uint32_t seq = 0;             // number of the last step issued on this staging buffer
    bool armed = false;           // step `seq` is enqueued behind a wait on flag
    uint64_t armed_sig = 0;       // everything the armed launches were made for (see step_sig)
    // the armed step's call, argument by argument: a call that repeats them byte for byte is released
    // before anything else is done (validation and planning then run while the GPU works)
    pkv_shape id_shape;
    pkv_split_policy id_policy;
    const void *id_k = nullptr, *id_v = nullptr, *id_out = nullptr, *id_ws = nullptr, *id_ds = nullptr, *id_stream = nullptr;
    float id_scale = 0.f;
    size_t id_scratch_bytes = 0, id_ws_bytes = 0;
    pkv_counters armed_counters;  // what the armed step's call will report
    uint64_t seen[32];            // launch keys that have been launched WITHOUT a pending wait (kernels loaded)
    int nseen = 0;
};
PipeCtx* pipe_ctx(void* staging, bool create) {
    thread_local PipeCtx table[8];
    thread_local int next = 0;
    for (PipeCtx& c : table)
        if (c.staging == staging && staging != nullptr) return &c;
    if (!create) return nullptr;
    // reuse a slot that holds no armed step
    for (int k = 0; k < 8; ++k) {
        PipeCtx& c = table[(next + k) % 8];
        if (!c.armed) {
            next = (next + k + 1) % 8;
            c = PipeCtx();
            c.staging = staging;
            return &c;
        }
    }
    return nullptr;
}

inline uint64_t mix64(uint64_t h, uint64_t v) {
    h ^= v + 0x9e3779b97f4a7c15ull + (h << 6) + (h >> 2);
    return h * 0xff51afd7ed558ccdull;
}
// What decides WHICH kernel instantiations run_decode launches: the decode kernel is <G, HG, d, dtype>
// with HG chosen from the host plan's (row, split) pairs (run_decode), the merge kernel <G, warps, slices>
// follows from the policy, B * Hq and d alone (launch_merge) and is launched when a row has two splits.
// Two steps with the same key launch the same instantiations.
uint64_t launch_key(const pkv_shape& s, const Resolved& rp, const QueueHeader& hdr, int sms) {
    uint64_t h = 0x706b7670697065ull;
    const int hg = choose_heads_per_cta(rp.heads_per_cta, s.Hkv, hdr.total_row_slots, sms, max_heads_per_cta(rp.G, s.d));
    const int64_t v[] = {s.B, s.Hq, s.Hkv, s.d, s.page_size, s.kv_dtype, rp.S, rp.tile_tokens, rp.split_mode, rp.chunk_tiles, rp.route,
                         rp.merge_mode, rp.kernel, rp.G, rp.num_sms, rp.flags, rp.heads_per_cta, rp.prefetch_kb, sms,
                         hg, hdr.max_row_splits > 1, hdr.num_tasks > 0};
    for (int64_t x : v) h = mix64(h, (uint64_t)x);
    return h;
}
// Everything an armed step was enqueued for, besides the lengths and the table (compared byte by byte).
uint64_t step_sig(uint64_t key, const pkv_shape& s, const QueueHeader& hdr, const void* k, const void* v, const void* out, const void* ws,
                  const void* ds, float scale, const void* stream) {
    uint64_t h = key;
    uint32_t sb;
    std::memcpy(&sb, &scale, 4);
    const uint64_t x[] = {(uint64_t)(uintptr_t)k, (uint64_t)(uintptr_t)v, (uint64_t)(uintptr_t)out, (uint64_t)(uintptr_t)ws,
                          (uint64_t)(uintptr_t)ds, (uint64_t)(uintptr_t)stream, sb, (uint64_t)s.max_pages, (uint64_t)s.num_pages,
                          (uint64_t)s.kv_stride_page, (uint64_t)s.kv_stride_token, (uint64_t)s.kv_stride_head,
                          (uint64_t)(uintptr_t)s.k_scale, (uint64_t)(uintptr_t)s.v_scale, (uint64_t)hdr.num_tasks};
    for (uint64_t y : x) h = mix64(h, y);
    return h;
}

// Block-table rows of `table` whose used entries differ from the shadow: counts the runs (and their
// bytes) without touching anything (apply = false), or copies them into the shadow and records them as
// pieces (apply = true).  Returns false when there are more runs than `cap` pieces.
struct Piece { size_t off, n; };
bool table_runs(const pkv_shape& s, const HostImage& im, unsigned char* hs, const int32_t* table, const int32_t* lens, bool fresh,
                bool apply, Piece* pieces, int cap, int* npieces, size_t* bytes) {
    int32_t* shadow = reinterpret_cast<int32_t*>(hs + im.block_table);
    int32_t run_lo = -1;
    auto flush = [&](int32_t hi) {
        if (run_lo < 0) return true;
        const size_t off = im.block_table + 4 * (size_t)run_lo * s.max_pages, n = 4 * (size_t)(hi - run_lo) * s.max_pages;
        run_lo = -1;
        *bytes += n;
        if (*npieces >= cap) return false;
        pieces[(*npieces)++] = Piece{off, n};
        return true;
    };
    for (int32_t i = 0; i < s.B; ++i) {
        const int64_t N = lens[i];
        const size_t used = N > 0 ? (size_t)((N + s.page_size - 1) / s.page_size) : 0;
        const int32_t* src = table + (size_t)i * s.max_pages;
        int32_t* dst = shadow + (size_t)i * s.max_pages;
        const bool changed = used > 0 && (fresh || std::memcmp(src, dst, 4 * used) != 0);
        if (changed) {
            if (apply) std::memcpy(dst, src, 4 * used);
            if (run_lo < 0) run_lo = i;
        } else if (!flush(i)) {
            return false;
        }
    }
    return flush(s.B);
}

// Spins until *word == want (a word the GPU writes into pinned host memory).  The stream is polled
// now and then so that a failed launch or a faulted kernel ends the wait with an error.
pkv_status spin_until(const volatile uint32_t* word, uint32_t want, cudaStream_t cs, const char* what) {
    for (uint64_t spins = 0;; ++spins) {
        if (*word == want) return PKV_OK;
        if ((spins & 0xffff) == 0xffff) {
            const cudaError_t e = cudaStreamQuery(cs);
            if (e != cudaSuccess && e != cudaErrorNotReady) return cuda_fail(e, what);
            if (e == cudaSuccess && *word != want) {      // the stream is idle and the word never came
                set_error("%s: the stream drained without the step's completion word (%u, want %u)", what, *word, want);
                return PKV_ERR_CUDA;
            }
        }
        if (spins > (1ull << 34)) { set_error("%s: timed out", what); return PKV_ERR_CUDA; }
#if defined(__x86_64__)
        __builtin_ia32_pause();
#endif
    }
}

}  // namespace
}  // namespace pkv

extern "C" {

size_t pkv_host_scratch_bytes(const pkv_shape* shape, const pkv_split_policy* policy) {
    Resolved rp;
    if (validate_and_resolve(shape, policy, 0, /*bound_ok=*/true, &rp) != PKV_OK) return 0;
    return host_image(*shape).total;
}

pkv_status pkv_decode_host(const pkv_shape* shape, const pkv_split_policy* policy, const void* q_host,
                           const void* k_cache_dev, const void* v_cache_dev, const int32_t* block_table_host,
                           const int32_t* seq_lens_host, void* out_host, float scale, void* host_staging,
                           void* dev_scratch, size_t scratch_bytes, void* workspace, size_t workspace_bytes,
                           void* stream, pkv_counters* counters_out) {
    clear_error();
    Resolved rp;
    const int sms = device_sm_count();
    pkv_status st = validate_and_resolve(shape, policy, sms, false, &rp);
    if (st != PKV_OK) return st;
    if (sms <= 0) { set_error("no CUDA device"); return PKV_ERR_CUDA; }
    {   // a step that pkv_decode_host_pipelined left armed on this staging buffer would block the stream for good
        const PipeCtx* pc = pipe_ctx(host_staging, false);
        if (pc && pc->armed) {
            st = pkv_decode_host_drain(host_staging, stream);
            if (st != PKV_OK) return st;
            clear_error();
        }
    }
    pkv_split_policy auto_pol;
    if (rp.auto_mode && seq_lens_host) {
        // PKV_SPLIT_AUTO: the cost model picks this step's policy from the host-resident lengths
        // ("for each decode step, the harness estimates T_r")
        st = auto_policy(*shape, *policy, seq_lens_host, sms, &auto_pol);
        if (st == PKV_OK) st = validate_and_resolve(shape, &auto_pol, sms, false, &rp);
        if (st != PKV_OK) return st;
    }
    const pkv_shape& s = *shape;
    if (s.B > 0 && (!q_host || !k_cache_dev || !v_cache_dev || !block_table_host || !seq_lens_host || !out_host)) {
        set_error("null pointer argument");
        return PKV_ERR_INVALID_ARG;
    }
    if (!host_staging || !dev_scratch || reinterpret_cast<uintptr_t>(dev_scratch) % 256) {
        set_error("host_staging / dev_scratch null or dev_scratch not 256-byte aligned");
        return PKV_ERR_INVALID_ARG;
    }
    const HostImage im = host_image(s);
    if (scratch_bytes < im.total) { set_error("scratch has %zu bytes, %zu needed", scratch_bytes, im.total); return PKV_ERR_WORKSPACE; }
    const WorkspaceLayout L = workspace_layout(s, rp.S);
    st = check_workspace(workspace, workspace_bytes, L);
    if (st != PKV_OK) return st;
    cudaStream_t cs = static_cast<cudaStream_t>(stream);
    // here the lengths ARE host-checkable; the page ids are checked when the caller asks for it
    for (int32_t i = 0; i < s.B; ++i) {
        const int64_t N = seq_lens_host[i];
        if (N > (int64_t)s.max_pages * s.page_size) {
            set_error("seq_lens[%d]=%lld exceeds max_pages*page_size=%lld", i, (long long)N, (long long)s.max_pages * s.page_size);
            return PKV_ERR_INVALID_ARG;
        }
        if (rp.flags & PKV_FLAG_VALIDATE) {
            const int64_t np = N > 0 ? (N + s.page_size - 1) / s.page_size : 0;
            for (int64_t j = 0; j < np; ++j) {
                const int32_t pg = block_table_host[(int64_t)i * s.max_pages + j];
                if (pg < 0 || pg >= s.num_pages) {
                    set_error("block_table[%d][%lld]=%d outside [0, %lld)", i, (long long)j, pg, (long long)s.num_pages);
                    return PKV_ERR_INVALID_ARG;
                }
            }
        }
    }

    // Host planning (planning is part of the serving-facing time): only the COUNTS of
    // the queue -- tasks, max_i n_i, (row, split) pairs -- which decide the launches (A13)
    // and the kernel's grid; the queue itself is derived inside the decode kernel from the uploaded
    // lengths (fused build), bit-identical to the host planner's.
    unsigned char* hs = static_cast<unsigned char*>(host_staging);
    unsigned char* ds = static_cast<unsigned char*>(dev_scratch);
    QueueHeader hdr_v;
    QueueHeader* hdr = &hdr_v;
    plan_host(s, rp, seq_lens_host, nullptr, 0, nullptr, nullptr, hdr);
    // seq_lens and q: through the staging image, one cudaMemcpyAsync.  (Letting the kernels read a
    // pinned q in place was measured and dropped: every split CTA re-reads its q slice in 4-byte
    // pieces over the host link -- config 2: 74.6 us per step against 43.4 staged.)
    const size_t q_bytes = 2 * (size_t)s.B * s.Hq * s.d;
    std::memcpy(hs + im.seq_lens, seq_lens_host, 4 * (size_t)s.B);
    std::memcpy(hs + im.q, q_host, q_bytes);
    size_t h2d = (im.q - im.seq_lens) + q_bytes;
    cudaError_t e = cudaMemcpyAsync(ds + im.seq_lens, hs + im.seq_lens, h2d, cudaMemcpyHostToDevice, cs);
    if (e != cudaSuccess) return cuda_fail(e, "H2D lengths and q");
    const void* q_dev = ds + im.q;
    const int32_t* lens_dev = reinterpret_cast<const int32_t*>(ds + im.seq_lens);
    // block table: rows whose used entries differ from the shadow (everything on first use)
    {
        StageHeader* sh = reinterpret_cast<StageHeader*>(hs + im.hdr);
        const bool fresh = sh->magic != kStageMagic || sh->B != s.B || sh->max_pages != s.max_pages || sh->dev != dev_scratch;
        int32_t* shadow = reinterpret_cast<int32_t*>(hs + im.block_table);
        int32_t run_lo = -1;       // pending run of changed rows [run_lo, i)
        auto flush = [&](int32_t hi) -> cudaError_t {
            if (run_lo < 0) return cudaSuccess;
            const size_t off = im.block_table + 4 * (size_t)run_lo * s.max_pages, n = 4 * (size_t)(hi - run_lo) * s.max_pages;
            run_lo = -1;
            h2d += n;
            return cudaMemcpyAsync(ds + off, hs + off, n, cudaMemcpyHostToDevice, cs);
        };
        for (int32_t i = 0; i < s.B; ++i) {
            const int64_t N = seq_lens_host[i];
            const size_t used = N > 0 ? (size_t)((N + s.page_size - 1) / s.page_size) : 0;
            const int32_t* src = block_table_host + (size_t)i * s.max_pages;
            int32_t* dst = shadow + (size_t)i * s.max_pages;
            const bool changed = used > 0 && (fresh || std::memcmp(src, dst, 4 * used) != 0);
            if (changed) {
                std::memcpy(dst, src, 4 * used);
                if (run_lo < 0) run_lo = i;
            } else if (run_lo >= 0) {
                e = flush(i);
                if (e != cudaSuccess) return cuda_fail(e, "H2D block table rows");
            }
        }
        e = flush(s.B);
        if (e != cudaSuccess) return cuda_fail(e, "H2D block table rows");
        sh->magic = kStageMagic; sh->B = s.B; sh->max_pages = s.max_pages; sh->table_src = block_table_host; sh->dev = dev_scratch;
    }

    WsPtrs ws = carve(workspace, L);
    int dl = 0, ml = 0;
    // Pinned (page-locked, device-mapped) out_host: a small kernel behind the merge stores the FP16 result
    // into it -- 8 KiB of posted writes per row -- and the copy-engine hop disappears from the step.
    // Pageable out_host: one cudaMemcpyAsync from dev_scratch.
    void* out_mapped = mapped_device_pointer(out_host, 16, (rp.flags & PKV_FLAG_OUT_PINNED) != 0);
    const bool zero_copy_out = out_mapped != nullptr;
    // the kernels write the result into the device image either way: a kernel that stores into host memory
    // itself cannot complete before those stores have drained over the link (measured on the pipelined step,
    // DESIGN.md 6.6); a small kernel chained behind them carries it to a pinned out_host
    void* out_dev = ds + im.out;
    const bool fused = rp.kernel == PKV_KERNEL_TMA_MMA && !(rp.flags & PKV_FLAG_SEPARATE_BUILD) && s.B <= kMaxFusedRows;
    if (!fused && hdr->num_tasks > 0) {
        e = launch_builder(s, rp, lens_dev, nullptr, ws.q.hdr, ws.q.split_offsets, ws.fuse_counters, ws.q.rowslots, ws.q.tasks,
                           L.slots_cap, cs);
        if (e != cudaSuccess) return cuda_fail(e, "builder launch");
    }
    st = run_decode(s, rp, q_dev, k_cache_dev, v_cache_dev, reinterpret_cast<const int32_t*>(ds + im.block_table),
                    lens_dev, nullptr, out_dev, nullptr, scale, nullptr, ws.q, ws, hdr->num_tasks, hdr->max_row_splits,
                    hdr->total_row_slots, sms, PKV_STAGE_ALL, fused, L.slots_cap, cs, &dl, &ml);
    if (st != PKV_OK) return st;
    const size_t out_bytes = 2 * (size_t)s.B * s.Hq * s.d;
    e = zero_copy_out ? launch_signal(nullptr, 0, !(rp.flags & PKV_FLAG_NO_PDL), ds + im.out, out_mapped, out_bytes, cs)
                      : cudaMemcpyAsync(out_host, ds + im.out, out_bytes, cudaMemcpyDeviceToHost, cs);
    if (e == cudaSuccess) e = cudaStreamSynchronize(cs);
    if (e != cudaSuccess) return cuda_fail(e, "D2H out / sync");
    if (counters_out) {
        std::memset(counters_out, 0, sizeof(*counters_out));
        counters_out->tasks = hdr->num_tasks;
        counters_out->empty_tasks = hdr->empty_tasks;
        counters_out->decode_launches = dl;
        counters_out->merge_launches = ml;
        counters_out->build_launches = (!fused && hdr->num_tasks > 0) ? 1 : 0;
        counters_out->useful_kv_bytes = hdr->sum_seq_lens * 2 * s.Hkv * s.d * (s.kv_dtype != PKV_KV_F16 ? 1 : 2);
        counters_out->merge_bytes = (int64_t)hdr->num_tasks * rp.G * (s.d + 2) * 4;
        counters_out->num_splits = hdr->resolved_splits;
        counters_out->max_row_splits = hdr->max_row_splits;
        counters_out->chunk_tiles = hdr->chunk_tiles;
        counters_out->h2d_bytes = (int64_t)h2d;
        counters_out->d2h_bytes = (int64_t)out_bytes;
        counters_out->launched_decode = dl;
        counters_out->launched_merge = ml;
    }
    return PKV_OK;
}

}  // extern "C"

// ------------------------------------------------------------------ pipelined host-buffer step

namespace pkv {
namespace {

struct PipeStep {          // one step's launches, as issue_step needs them
    Resolved rp;
    QueueHeader hdr;
    const void* k;
    const void* v;
    void* out_dev;
    Piece pieces[kMaxStageSegs];
    int npieces;
    size_t h2d;
};

void fill_counters(const pkv_shape& s, const PipeStep& st, int dl, int ml, pkv_counters* c) {
    std::memset(c, 0, sizeof(*c));
    c->tasks = st.hdr.num_tasks;
    c->empty_tasks = st.hdr.empty_tasks;
    c->decode_launches = dl;
    c->merge_launches = ml;
    c->useful_kv_bytes = st.hdr.sum_seq_lens * 2 * s.Hkv * s.d * (s.kv_dtype != PKV_KV_F16 ? 1 : 2);
    c->merge_bytes = (int64_t)st.hdr.num_tasks * st.rp.G * (s.d + 2) * 4;
    c->num_splits = st.hdr.resolved_splits;
    c->max_row_splits = st.hdr.max_row_splits;
    c->chunk_tiles = st.hdr.chunk_tiles;
    c->h2d_bytes = (int64_t)st.h2d;
    c->d2h_bytes = (int64_t)2 * s.B * s.Hq * s.d;
    c->launched_decode = dl;
    c->launched_merge = ml;
}

// gate / stage kernel [waits until the host releases step `seq`] -> decode -> merge -> signal (done word).
pkv_status issue_step(const pkv_shape& s, const PipeStep& st, uint32_t seq, bool gate, float scale, const HostImage& im,
                      const void* hs_mapped, unsigned char* ds, void* workspace, int sms, cudaStream_t cs, pkv_counters* counters) {
    uint32_t* words = reinterpret_cast<uint32_t*>(reinterpret_cast<uintptr_t>(hs_mapped) + im.hdr + kPipeWordsOffset);
    StageSegs segs = {};
    for (int k = 0; k < st.npieces; ++k) {
        // widened to 16-byte boundaries: the image and the scratch hold the same bytes around a changed
        // table row (its neighbours were uploaded from this very shadow; regions are 256-byte aligned)
        const size_t lo = st.pieces[k].off & ~(size_t)15, hi = (st.pieces[k].off + st.pieces[k].n + 15) & ~(size_t)15;
        segs.off[k] = (uint32_t)lo;
        segs.chunks[k] = (uint32_t)((hi - lo) / 16);
    }
    segs.n = st.npieces;
    cudaError_t e = launch_stage(hs_mapped, ds, segs, words, seq, gate, kGateTimeoutNs, cs);
    if (e != cudaSuccess) return cuda_fail(e, "stage kernel launch");
    const WorkspaceLayout L = workspace_layout(s, st.rp.S);
    const WsPtrs ws = carve(workspace, L);
    int dl = 0, ml = 0;
    // the result goes to the device image; the signal kernel takes it to the pinned out_host with the done word
    // (a kernel that writes host memory itself cannot complete before those writes have drained over the link)
    const pkv_status rs = run_decode(s, st.rp, ds + im.q, st.k, st.v, reinterpret_cast<const int32_t*>(ds + im.block_table),
                                     reinterpret_cast<const int32_t*>(ds + im.seq_lens), nullptr, ds + im.out, nullptr, scale, nullptr, ws.q, ws,
                                     st.hdr.num_tasks, st.hdr.max_row_splits, st.hdr.total_row_slots, sms, PKV_STAGE_ALL, true,
                                     L.slots_cap, cs, &dl, &ml);
    if (rs != PKV_OK) return rs;
    e = launch_signal(words, seq, !(st.rp.flags & PKV_FLAG_NO_PDL), ds + im.out, st.out_dev, 2 * (size_t)s.B * s.Hq * s.d, cs);
    if (e != cudaSuccess) return cuda_fail(e, "signal kernel launch");
    fill_counters(s, st, dl, ml, counters);
    return PKV_OK;
}

void release_step(PipeWords* w, uint32_t seq) {
    __atomic_thread_fence(__ATOMIC_RELEASE);      // the image's bytes before the flag
    *reinterpret_cast<volatile uint32_t*>(&w->flag) = seq;
    __atomic_thread_fence(__ATOMIC_SEQ_CST);
}

}  // namespace
}  // namespace pkv

extern "C" {

pkv_status pkv_decode_host_drain(void* host_staging, void* stream) {
    using namespace pkv;
    clear_error();
    PipeCtx* c = pipe_ctx(host_staging, false);
    if (!c || !c->armed) return PKV_OK;
    PipeWords* w = reinterpret_cast<PipeWords*>(static_cast<unsigned char*>(host_staging) + kPipeWordsOffset);
    release_step(w, c->seq);
    const pkv_status st = spin_until(&w->done, c->seq, static_cast<cudaStream_t>(stream), "pkv_decode_host_drain");
    c->armed = false;
    return st;
}

pkv_status pkv_decode_host_pipelined(const pkv_shape* shape, const pkv_split_policy* policy, const void* q_host,
                                     const void* k_cache_dev, const void* v_cache_dev, const int32_t* block_table_host,
                                     const int32_t* seq_lens_host, void* out_host, float scale, void* host_staging, void* dev_scratch,
                                     size_t scratch_bytes, void* workspace, size_t workspace_bytes, void* stream,
                                     const pkv_next_step* next, pkv_counters* counters_out) {
    using namespace pkv;
    clear_error();
    // Early release: the call repeats, byte for byte, the arguments the armed step was enqueued for.
    bool early = false;
    if (shape && policy && q_host && seq_lens_host && block_table_host) {
        PipeCtx* c0 = pipe_ctx(host_staging, false);
        if (c0 && c0->armed && std::memcmp(&c0->id_shape, shape, sizeof(*shape)) == 0 &&
            std::memcmp(&c0->id_policy, policy, sizeof(*policy)) == 0 && c0->id_k == k_cache_dev && c0->id_v == v_cache_dev &&
            c0->id_out == out_host && c0->id_ws == workspace && c0->id_ds == dev_scratch && c0->id_stream == stream &&
            std::memcmp(&c0->id_scale, &scale, 4) == 0 && c0->id_scratch_bytes == scratch_bytes && c0->id_ws_bytes == workspace_bytes) {
            const pkv_shape& s0 = *shape;
            const HostImage im0 = host_image(s0);
            unsigned char* hs0 = static_cast<unsigned char*>(host_staging);
            PipeWords* w0 = reinterpret_cast<PipeWords*>(hs0 + im0.hdr + kPipeWordsOffset);
            Piece tmp[1];
            int nrun = 0;
            size_t run_bytes = 0;
            if (*reinterpret_cast<volatile uint32_t*>(&w0->expired) != c0->seq &&
                std::memcmp(hs0 + im0.seq_lens, seq_lens_host, 4 * (size_t)s0.B) == 0 &&
                table_runs(s0, im0, hs0, block_table_host, seq_lens_host, false, false, tmp, 0, &nrun, &run_bytes) && run_bytes == 0) {
                std::memcpy(hs0 + im0.q, q_host, 2 * (size_t)s0.B * s0.Hq * s0.d);
                release_step(w0, c0->seq);
                early = true;
            }
        }
    }
    auto plain = [&]() -> pkv_status {       // anything the pipeline cannot do: the synchronous call, after emptying the pipeline
        const pkv_status ds = pkv_decode_host_drain(host_staging, stream);
        if (ds != PKV_OK) return ds;
        return pkv_decode_host(shape, policy, q_host, k_cache_dev, v_cache_dev, block_table_host, seq_lens_host, out_host, scale,
                               host_staging, dev_scratch, scratch_bytes, workspace, workspace_bytes, stream, counters_out);
    };
    Resolved rp;
    const int sms = device_sm_count();
    if (!shape || !policy || sms <= 0 || validate_and_resolve(shape, policy, sms, false, &rp) != PKV_OK) return plain();
    const pkv_shape& s = *shape;
    if (s.B <= 0 || !q_host || !k_cache_dev || !v_cache_dev || !block_table_host || !seq_lens_host || !out_host || !host_staging ||
        !dev_scratch || reinterpret_cast<uintptr_t>(dev_scratch) % 256 || reinterpret_cast<uintptr_t>(host_staging) % 256)
        return plain();
    pkv_split_policy auto_pol;
    if (rp.auto_mode) {
        if (auto_policy(s, *policy, seq_lens_host, sms, &auto_pol) != PKV_OK || validate_and_resolve(shape, &auto_pol, sms, false, &rp) != PKV_OK)
            return plain();
    }
    const HostImage im = host_image(s);
    const bool cache_ptrs = (rp.flags & PKV_FLAG_OUT_PINNED) != 0;
    const void* hs_mapped = mapped_device_pointer(host_staging, 256, cache_ptrs);
    void* out_dev = mapped_device_pointer(out_host, 16, cache_ptrs);
    const bool can = hs_mapped && out_dev && rp.kernel == PKV_KERNEL_TMA_MMA &&
                     !(rp.flags & (PKV_FLAG_SEPARATE_BUILD | PKV_FLAG_VALIDATE)) && s.B <= kMaxFusedRows && scratch_bytes >= im.total &&
                     check_workspace(workspace, workspace_bytes, workspace_layout(s, rp.S)) == PKV_OK;
    PipeCtx* c = can ? pipe_ctx(host_staging, true) : nullptr;
    if (!c) return plain();
    for (int32_t i = 0; i < s.B; ++i)
        if ((int64_t)seq_lens_host[i] > (int64_t)s.max_pages * s.page_size) return plain();     // the plain call reports it

    cudaStream_t cs = static_cast<cudaStream_t>(stream);
    unsigned char* hs = static_cast<unsigned char*>(host_staging);
    unsigned char* ds = static_cast<unsigned char*>(dev_scratch);
    PipeWords* w = reinterpret_cast<PipeWords*>(hs + im.hdr + kPipeWordsOffset);
    StageHeader* sh = reinterpret_cast<StageHeader*>(hs + im.hdr);
    const bool fresh = sh->magic != kStageMagic || sh->B != s.B || sh->max_pages != s.max_pages || sh->dev != dev_scratch;
    if (c->seq == 0) {       // first step of this pipeline: nothing of it is in flight
        w->flag = 0; w->staged = 0; w->done = 0; w->expired = 0;
    }
    const size_t q_bytes = 2 * (size_t)s.B * s.Hq * s.d;
    const size_t head_bytes = (im.q - im.seq_lens) + q_bytes;       // lengths and q: one piece

    PipeStep cur;
    cur.rp = rp; cur.k = k_cache_dev; cur.v = v_cache_dev; cur.out_dev = out_dev;
    plan_host(s, rp, seq_lens_host, nullptr, 0, nullptr, nullptr, &cur.hdr);
    const uint64_t key = launch_key(s, rp, cur.hdr, sms);
    const uint64_t sig = step_sig(key, s, cur.hdr, k_cache_dev, v_cache_dev, out_dev, workspace, dev_scratch, scale, stream);
    pkv_counters counters;
    uint32_t my_seq = 0;
    bool was_armed = false;
    if (c->armed) {
        // Was the armed step made for exactly this call?  Same launches and buffers, same lengths, no table change.
        Piece tmp[1];
        int nrun = 0;
        size_t run_bytes = 0;
        const bool same = !fresh && c->armed_sig == sig && w->expired != c->seq &&
                          std::memcmp(hs + im.seq_lens, seq_lens_host, 4 * (size_t)s.B) == 0 &&
                          table_runs(s, im, hs, block_table_host, seq_lens_host, false, false, tmp, 0, &nrun, &run_bytes) && run_bytes == 0;
        if (same || early) {     // (early: released at the top of the call; the same comparisons, on the raw arguments)
            my_seq = c->seq;
            was_armed = true;
            if (!early) {
                std::memcpy(hs + im.q, q_host, q_bytes);
                release_step(w, my_seq);
            }
            counters = c->armed_counters;
            counters.armed_step = 1;
            c->armed = false;
        } else {
            // not the step that was predicted: it runs on what the image holds, its result is overwritten below
            const pkv_status st = pkv_decode_host_drain(host_staging, stream);
            if (st != PKV_OK) return st;
        }
    }
    if (my_seq == 0) {
        // issue this step without a wait: its inputs are in the image before anything is enqueued
        cur.npieces = 1;
        cur.pieces[0] = Piece{im.seq_lens, head_bytes};
        cur.h2d = head_bytes;
        Piece dry[kMaxStageSegs];
        int nrun = 0;
        size_t run_bytes = 0;
        if (cur.hdr.num_tasks == 0 ||
            !table_runs(s, im, hs, block_table_host, seq_lens_host, fresh, false, dry, kMaxStageSegs - 1, &nrun, &run_bytes) ||
            head_bytes + run_bytes > kMaxStageBytes)
            return plain();      // (nothing was modified)
        std::memcpy(hs + im.seq_lens, seq_lens_host, 4 * (size_t)s.B);
        std::memcpy(hs + im.q, q_host, q_bytes);
        nrun = 0;
        run_bytes = 0;
        table_runs(s, im, hs, block_table_host, seq_lens_host, fresh, true, cur.pieces + 1, kMaxStageSegs - 1, &nrun, &run_bytes);
        cur.npieces = 1 + nrun;
        cur.h2d += run_bytes;
        sh->magic = kStageMagic; sh->B = s.B; sh->max_pages = s.max_pages; sh->table_src = block_table_host; sh->dev = dev_scratch;
        __atomic_thread_fence(__ATOMIC_SEQ_CST);
        my_seq = ++c->seq;
        const pkv_status st = issue_step(s, cur, my_seq, false, scale, im, hs_mapped, ds, workspace, sms, cs, &counters);
        if (st != PKV_OK) return st;
        bool known = false;
        for (int k = 0; k < c->nseen; ++k) known = known || c->seen[k] == key;
        if (!known) { c->seen[c->nseen % 32] = key; c->nseen = c->nseen < 32 ? c->nseen + 1 : 32; }
    }

    // The stage kernel has read the image: the next step can be put into it and enqueued behind a wait
    // on the flag while the GPU works on this one.
    pkv_status st = spin_until(&w->staged, my_seq, cs, "pkv_decode_host_pipelined (stage)");
    if (st != PKV_OK) return st;
    if (next && next->seq_lens_host && next->block_table_host) {
        PipeStep nx;
        nx.rp = rp;
        bool ok = true;
        pkv_split_policy next_pol;
        Resolved base_rp;
        if (validate_and_resolve(shape, policy, sms, false, &base_rp) == PKV_OK && base_rp.auto_mode)
            ok = auto_policy(s, *policy, next->seq_lens_host, sms, &next_pol) == PKV_OK &&
                 validate_and_resolve(shape, &next_pol, sms, false, &nx.rp) == PKV_OK;
        for (int32_t i = 0; ok && i < s.B; ++i) ok = (int64_t)next->seq_lens_host[i] <= (int64_t)s.max_pages * s.page_size;
        ok = ok && check_workspace(workspace, workspace_bytes, workspace_layout(s, nx.rp.S)) == PKV_OK;
        nx.k = next->k_cache_dev ? next->k_cache_dev : k_cache_dev;
        nx.v = next->v_cache_dev ? next->v_cache_dev : v_cache_dev;
        nx.out_dev = next->out_host ? mapped_device_pointer(next->out_host, 16, cache_ptrs) : out_dev;
        ok = ok && nx.out_dev != nullptr;
        uint64_t nkey = 0;
        if (ok) {
            plan_host(s, nx.rp, next->seq_lens_host, nullptr, 0, nullptr, nullptr, &nx.hdr);
            nkey = launch_key(s, nx.rp, nx.hdr, sms);
            bool known = false;       // only kernels that have run before: loading a module under a pending wait would block
            for (int k = 0; k < c->nseen; ++k) known = known || c->seen[k] == nkey;
            ok = known && nx.hdr.num_tasks > 0;
        }
        Piece dry[kMaxStageSegs];
        int nrun = 0;
        size_t run_bytes = 0;
        ok = ok && table_runs(s, im, hs, next->block_table_host, next->seq_lens_host, false, false, dry, kMaxStageSegs - 1, &nrun, &run_bytes) &&
             head_bytes + run_bytes <= kMaxStageBytes;
        if (ok) {
            std::memcpy(hs + im.seq_lens, next->seq_lens_host, 4 * (size_t)s.B);
            nx.pieces[0] = Piece{im.seq_lens, head_bytes};
            nrun = 0;
            run_bytes = 0;
            table_runs(s, im, hs, next->block_table_host, next->seq_lens_host, false, true, nx.pieces + 1, kMaxStageSegs - 1, &nrun, &run_bytes);
            nx.npieces = 1 + nrun;
            nx.h2d = head_bytes + run_bytes;
            sh->table_src = next->block_table_host;
            const uint32_t nseq = ++c->seq;
            st = issue_step(s, nx, nseq, true, scale, im, hs_mapped, ds, workspace, sms, cs, &c->armed_counters);
            if (st != PKV_OK) return st;
            c->armed = true;
            c->id_shape = s; c->id_policy = *policy; c->id_k = nx.k; c->id_v = nx.v;
            c->id_out = next->out_host ? next->out_host : out_host;
            c->id_ws = workspace; c->id_ds = dev_scratch; c->id_stream = stream; c->id_scale = scale;
            c->id_scratch_bytes = scratch_bytes; c->id_ws_bytes = workspace_bytes;
            c->armed_sig = step_sig(nkey, s, nx.hdr, nx.k, nx.v, nx.out_dev, workspace, dev_scratch, scale, stream);
        }
    }
    st = spin_until(&w->done, my_seq, cs, "pkv_decode_host_pipelined (done)");
    if (st != PKV_OK) return st;
    // the gate gave up just as the step was being released: its inputs may have been stale -- do the step again
    if (was_armed && *reinterpret_cast<volatile uint32_t*>(&w->expired) == my_seq) return plain();
    if (counters_out) *counters_out = counters;
    return PKV_OK;
}

}  // extern "C"

