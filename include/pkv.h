/*
 * pkv.h -- C ABI of libpkv: paged GQA decode attention for B200 (sm_100a).
 *
 * The hot path of arxiv/paper_2606_26666 ("PersistentKV"): single-query grouped-query decode
 * attention that reads FP16 K/V through a native paged block table (sec. 3.2),
 * splits each row's sequence into split-local online-softmax states (sec. 3.3),
 * merges them exactly and launches only the non-empty (row, KV head, split)
 * tasks of a ragged batch through a compact workqueue (sec. 3.4).
 *
 * Conventions
 *   - plain C, no torch / C++ types.  "dev" pointers are CUDA device pointers, "host" pointers
 *     are ordinary host memory.  `stream` is a cudaStream_t passed as void* (NULL = legacy
 *     default stream).
 *   - the CALLER OWNS EVERY BUFFER (q, caches, tables, out, workspace).  pkv_build_workqueue,
 *     pkv_decode and pkv_merge never allocate, never synchronise and never read device data
 *     on the host, so all three may be captured into a CUDA graph.
 *   - the first pkv_workspace_init_bytes() bytes of a workspace (the queue header and the
 *     completion counters, all self-resetting) must be ZERO when the workspace is first used; the
 *     library keeps them consistent from then on.
 *   - every call returns a pkv_status; nothing throws or aborts.  pkv_last_error() gives a
 *     thread-local description of the last non-OK status.
 *   - host-checkable arguments are rejected before any launch.  Device-resident values
 *     (seq_lens[i] > max_pages*page_size, a page id >= num_pages) cannot be checked without a
 *     synchronisation: they are undefined behaviour -- unless policy.flags has PKV_FLAG_VALIDATE,
 *     which adds device-side checks that record the fault in the workspace's error word
 *     (pkv_counters.error_word) and keep the kernels inside the caller's buffers (PAPER.md:67:
 *     every bound is derived from N_i).  seq_lens[i] == 0 is legal: the row emits no task,
 *     out[i] = 0 and lse[i] = -inf (reading A9).
 *   - compiled-in shapes: G = Hq/Hkv in {1, 2, 4, 8, 16}, page_size in {16, 32, 64}, d = 128; d in
 *     {64, 256} (FP16 caches) and one-byte caches (FP8 E4M3, INT8; d = 128) on the TMA kernel; the
 *     fused KV-append for d = 128.  Anything else returns PKV_ERR_UNSUPPORTED.
 */
#ifndef PKV_H_
#define PKV_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(_WIN32)
#define PKV_API
#else
#define PKV_API __attribute__((visibility("default")))
#endif

typedef enum {
    PKV_OK = 0,
    PKV_ERR_INVALID_ARG = 1,  /* null pointer, negative size, Hq % Hkv, misaligned pointer/stride */
    PKV_ERR_UNSUPPORTED = 2,  /* shape / G / arch not compiled in                                */
    PKV_ERR_WORKSPACE = 3,    /* caller workspace smaller than pkv_workspace_bytes()             */
    PKV_ERR_CUDA = 4          /* CUDA runtime / driver error; see pkv_last_error()               */
} pkv_status;

typedef enum { PKV_ROUTE_RECT = 0, PKV_ROUTE_WORKQUEUE = 1 } pkv_route;
typedef enum { PKV_MERGE_SEPARATE = 0, PKV_MERGE_FUSED = 1 } pkv_merge_mode;
typedef enum { PKV_SPLIT_FIXED_COUNT = 0, PKV_SPLIT_FIXED_CHUNK = 1, PKV_SPLIT_BALANCED = 2, PKV_SPLIT_AUTO = 3 } pkv_split_mode;
/* which decode kernel runs the tile loop */
typedef enum {
    PKV_KERNEL_AUTO = 0, /* = PKV_KERNEL_TMA_MMA                                                 */
    PKV_KERNEL_TMA_MMA = 1, /* TMA page loads -> mbarrier ring -> ldmatrix + HMMA, warp-specialised */
    PKV_KERNEL_SIMT = 2  /* 16-byte vector loads straight from global, FP32 FFMA + warp shuffles */
} pkv_kernel;

/*
 * Split policy (PAPER.md:63-67 row-local bounds; PAPER.md:89 split policy).  All bounds are in
 * tiles of `tile_tokens` tokens, counted from the row's true length N_i = seq_lens[i]:
 *   T_i = ceil(N_i / tile_tokens)
 *   FIXED_COUNT: S_i = S                          (S = num_splits, or the auto rule when 0)
 *   FIXED_CHUNK: S_i = min(S, ceil(T_i / chunk_tiles))   (S = num_splits, or 256 when 0)
 *   c_i = ceil(T_i / S_i), n_i = ceil(T_i / c_i); split s of row i covers tiles
 *   [s*c_i, min((s+1)*c_i, T_i)), s = 0 .. n_i-1                      (reading A6)
 * Auto rule (A12): S = clamp(ceil(4*num_sms / (B*Hkv)), 1, 256).
 *   BALANCED: FIXED_CHUNK whose chunk_tiles is derived from the whole batch's true lengths
 *   ("CTA-work and length-based tile bounds"; per-row split counts, PAPER.md:271;
 *   DESIGN.md reading A21).  With U = num_sms, W = sum_i T_i, m = ceil(256 / tile_tokens):
 *     c2 = max(m, ceil(W / (32*U)))                   (many waves: about 32 pairs per SM,
 *                                                       handed out dynamically)
 *     single wave: the smallest c in [ceil(W/U), ceil(W/U) + c2] with
 *                  sum_i ceil(T_i / c) <= U   (every SM gets at most one (row, split) pair and
 *                  the busiest SM's share exceeds the mean W/U by at most one many-wave chunk);
 *     chunk = that c if it exists, else c2.
 *   chunk_tiles of the policy is ignored; S = num_splits (256 when 0) still caps n_i.
 *   AUTO: the cost model decides.  pkv_decode_host, where the lengths are on the
 *   host, runs pkv_choose_policy with the default B200 constants before every step; calls whose
 *   lengths are device-resident (pkv_decode, pkv_build_workqueue) and the pure sizing functions
 *   treat AUTO as BALANCED, the candidate that needs no host knowledge of the lengths.
 */
typedef struct {
    int32_t tile_tokens; /* > 0, multiple of page_size; the paper uses 32          */
    int32_t split_mode;  /* pkv_split_mode                                                       */
    int32_t num_splits;  /* >= 0, <= 256; see above                                              */
    int32_t chunk_tiles; /* FIXED_CHUNK: tiles per task (> 0)                                    */
    int32_t route;       /* pkv_route                                                            */
    int32_t merge_mode;  /* pkv_merge_mode                                                       */
    int32_t num_sms;     /* SM count for the auto rule and for BALANCED; 0 = the current device's
                            (device calls only; the host builder needs it > 0 then)             */
    int32_t kernel;      /* pkv_kernel                                                           */
    int32_t flags;       /* bit set of pkv_flag                                                  */
    int32_t heads_per_cta; /* TMA kernel: KV heads one CTA streams together:
                            0 = automatic (the largest of 8/4/2/1 dividing Hkv that leaves one work
                            unit per SM), else 1, 2, 4 or 8 and a divisor of Hkv                  */
    int32_t prefetch_kb; /* TMA kernel: KiB of its first work unit's K/V that every CTA requests into
                            L2 BEFORE its dependency wait (programmatic launch; DESIGN.md "L2
                            prefetch"): 0 = library default, < 0 = off                            */
} pkv_split_policy;

/* policy.flags */
typedef enum {
    /* Device-side validation of device-resident inputs (SURVEY.md sec. 8(b) debug check): a row
     * with seq_lens[i] > max_pages*page_size is decoded as if its length were max_pages*page_size
     * and sets PKV_DEVERR_SEQ_LEN; a block-table entry outside [0, num_pages) that a task would
     * dereference is replaced by page 0 and sets PKV_DEVERR_PAGE_ID.  The kernels then never read
     * outside the block table or the page pool; the result of a faulted row is unspecified. */
    PKV_FLAG_VALIDATE = 1,
    /* Launch the kernels of this call without programmatic dependent launch: every
     * kernel then starts after its predecessor in the stream has finished. */
    PKV_FLAG_NO_PDL = 2,
    /* Run the workqueue builder as its own kernel even where the TMA decode kernel could derive the
     * queue itself. */
    PKV_FLAG_SEPARATE_BUILD = 4,
    /* Test only: the TMA decode kernel discards the plan it made speculatively before its dependency
     * wait and plans again afterwards -- the path taken when the kernel right before pkv_decode wrote
     * seq_lens. */
    PKV_FLAG_TEST_REPLAN = 8,
    /* pkv_decode_host: the caller promises that out_host is pinned, device-mapped host memory that
     * stays registered while it is passed to the library.  The device address is then looked up once
     * per buffer (per thread) instead of in every call (a pointer query costs about a microsecond).
     * Without the flag every call asks the driver, so a buffer that was freed and whose address was
     * reused can never be mistaken for a mapped one. */
    PKV_FLAG_OUT_PINNED = 16
} pkv_flag;
/* bits of pkv_counters.error_word (sticky in the workspace until its init bytes are zeroed again) */
typedef enum { PKV_DEVERR_QUEUE_OVERFLOW = 1, PKV_DEVERR_SEQ_LEN = 2, PKV_DEVERR_PAGE_ID = 4 } pkv_device_error;

/* One workqueue entry: tile interval [t_begin, t_end) of row `row`, KV head `kvh`;
 * token range = [t_begin*tile_tokens, min(t_end*tile_tokens, N_row)). */
typedef struct { int32_t row, kvh, split, t_begin, t_end; } pkv_task;

/*
 * Problem shape.  Caches are FP16 buffers addressed as
 *   elem(page, token, head, c) = page*kv_stride_page + token*kv_stride_token + head*kv_stride_head + c
 * (strides in elements, c is unit-stride).  All three strides 0 = the default layout
 * [num_pages, page_size, Hkv, d] (BASELINE.json north_star; reading A1); the paper's
 * [num_pages, Hkv, page_size, d] is kv_stride_head = page_size*d,
 * kv_stride_token = d.  Strides must be multiples of 8 elements (16 bytes).
 */
typedef struct {
    int32_t B, Hq, Hkv, d, page_size, max_pages; /* block_table is [B, max_pages] int32          */
    int64_t num_pages;
    int64_t kv_stride_page, kv_stride_token, kv_stride_head;
    /* FP8 KV cache with in-loop dequantisation ("dequantization-aware paged decode";
     * DESIGN.md reading A28): kv_dtype = PKV_KV_E4M3 / PKV_KV_INT8 makes k_cache / v_cache buffers of
     * OCP FP8 E4M3 / two's-complement INT8 bytes (same layout, strides in elements = bytes, multiples
     * of 16) that stand for
     *   k = k_scale[kv head] * dec(byte),  v = v_scale[kv head] * dec(byte)
     * k_scale / v_scale: dev float [Hkv], or NULL for 1.0.  q and out stay FP16, arithmetic as for
     * FP16 caches (E4M3 values are FP16 numbers).  TMA kernel, d = 128 only. */
    int32_t kv_dtype;                            /* pkv_kv_dtype; 0 = FP16                       */
    int32_t reserved_;
    const float* k_scale;
    const float* v_scale;
} pkv_shape;
typedef enum { PKV_KV_F16 = 0, PKV_KV_E4M3 = 1, PKV_KV_INT8 = 2 } pkv_kv_dtype;

/* Scheduler-derived counters with the definitions of Table 4 (A13,
 * A14).  Filled by pkv_get_counters from the workqueue state of the last build / decode. */
typedef struct {
    int64_t tasks;           /* non-empty tasks (workqueue) or B*Hkv*S grid cells (rect)         */
    int64_t empty_tasks;     /* rect route only: grid cells with an empty tile interval          */
    int64_t decode_launches; /* 1, or 0 when there is no task                                    */
    int64_t merge_launches;  /* 1 if a separate merge kernel is needed, else 0                   */
    int64_t build_launches;  /* device builder kernel launches (the paper builds on the host)    */
    int64_t useful_kv_bytes; /* sum_i N_i * 2*Hkv*d*2                                            */
    int64_t merge_bytes;     /* partial slots * G * (d+2) * 4 (one pass)                         */
    int64_t num_splits;      /* resolved S                                                       */
    int64_t max_row_splits;  /* max_i n_i                                                        */
    int64_t chunk_tiles;     /* FIXED_CHUNK / BALANCED: resolved tiles per task; else 0          */
    int64_t h2d_bytes;       /* pkv_decode_host only: bytes copied host->device this step        */
    int64_t d2h_bytes;       /* pkv_decode_host only: bytes copied device->host this step        */
    /* What the last build / decode on this workspace REALLY launched (each kernel leaves its mark
     * in the queue header).  On the device path the host cannot see the lengths, so a merge kernel
     * is launched whenever the policy allows more than one split per row, and a decode kernel
     * even when every row is empty: these can exceed the scheduler-derived counts above. */
    int64_t launched_build, launched_decode, launched_merge;
    int64_t error_word;      /* bit set of pkv_device_error                                      */
    int64_t armed_step;      /* pkv_decode_host_pipelined only: 1 = this step's launches had been
                                enqueued by the previous call and were only released by this one */
} pkv_counters;

/* Library/ABI version: (major << 16) | minor. */
PKV_API int32_t pkv_version(void);
/* Thread-local text of the last error on this thread ("" if none).  Never NULL. */
PKV_API const char* pkv_last_error(void);

/* Bytes of device workspace pkv_build_workqueue / pkv_decode need for this shape and policy.
 * Pure function (no CUDA call).  Returns 0 on invalid arguments.  With num_splits == 0 and
 * num_sms == 0 the bound for S = 256 is returned. */
PKV_API size_t pkv_workspace_bytes(const pkv_shape* shape, const pkv_split_policy* policy);
/* Leading bytes of the workspace the caller must zero once before first use (a few hundred bytes +
 * 4*B*Hkv).  Pure function; 0 on invalid arguments. */
PKV_API size_t pkv_workspace_init_bytes(const pkv_shape* shape, const pkv_split_policy* policy);

/* Split-bound policy + compact workqueue on the HOST.  Pure CPU, no CUDA.
 * seq_lens_host [B].  Writes at most tasks_cap tasks in canonical order (row, kvh, split --
 * DESIGN.md A7), split_offsets_out [B+1] = exclusive prefix sum of n_i (workqueue route) or of
 * S (rect route), *num_tasks_out.  PKV_ERR_WORKSPACE if tasks_cap is too small (then
 * *num_tasks_out holds the needed count).  tasks_out may be NULL with tasks_cap == 0 to count. */
PKV_API pkv_status pkv_build_workqueue_host(const pkv_shape* shape, const pkv_split_policy* policy,
                                            const int32_t* seq_lens_host, pkv_task* tasks_out,
                                            int32_t tasks_cap, int32_t* split_offsets_out,
                                            int32_t* num_tasks_out);

/* The same, by one kernel on the DEVICE into the (private) workspace; seq_lens_dev [B] is read
 * by the kernel only.  Marks the workspace's queue as built for the next pkv_decode. */
PKV_API pkv_status pkv_build_workqueue(const pkv_shape* shape, const pkv_split_policy* policy,
                                       const int32_t* seq_lens_dev, void* workspace,
                                       size_t workspace_bytes, void* stream);

/*
 * One decode step (Eq. 1 through the block table, split per `policy`).
 *   q           dev [B, Hq, d] f16          k_cache, v_cache  dev, see pkv_shape
 *   block_table dev [B, max_pages] i32      seq_lens          dev [B] i32
 *   out         dev [B, Hq, d] f16          lse               dev [B, Hq] f32 or NULL
 *   scale       <= 0 means 1/sqrt(d)        (natural-log LSE of the scaled scores)
 * build_queue != 0: runs the device builder first (as pkv_build_workqueue); 0: uses the queue
 * already in `workspace` (built for the same shape/policy and the same seq_lens values).
 * Launches: [builder] + decode + [merge].  With the TMA kernel and B <= 512 the decode kernel
 * derives the queue from seq_lens itself ("fused build": no builder launch; the queue is still
 * written to the workspace, bit-identical to pkv_build_workqueue's).  The merge launch is skipped
 * when the policy cannot produce more than one split per row, or merge_mode is FUSED.
 * Results are bitwise reproducible from launch to launch for the same inputs, policy and device.
 * Programmatic launch: the decode kernel may start while the kernel before it in the stream is
 * still running.  It then reads nothing but seq_lens (race-tolerant loads, for a speculative
 * plan) before that kernel has finished, and re-validates those lengths afterwards -- a
 * predecessor that writes seq_lens, q, the block table or the caches is handled correctly.
 * Heads per CTA: the TMA kernel streams HG = 8, 4, 2 or 1 KV heads per CTA (at most 4 with G = 16 or
 * d = 256), the largest value that still leaves work units for 85 % of the SMs given the bound B*S on
 * the (row, split) pairs; with
 * BALANCED the bound is policy.num_sms, so num_sms = SMs*HG/Hkv asks for HG heads per CTA
 * (policy.heads_per_cta overrides the choice).
 * L2 prefetch: before its dependency wait a CTA of the TMA kernel also asks the memory system to
 * bring the first policy.prefetch_kb KiB of its first work unit's K/V (found through the speculative
 * plan and a race-tolerant look at the block table) into L2.  A prefetch moves no data into the
 * program: L2 is the point of coherence, so whatever the predecessor kernel still writes is seen by
 * the loads after the wait; a wrong guess only costs bandwidth.
 */
PKV_API pkv_status pkv_decode(const pkv_shape* shape, const pkv_split_policy* policy, const void* q,
                              const void* k_cache, const void* v_cache, const int32_t* block_table,
                              const int32_t* seq_lens, void* out, float* lse, float scale,
                              int32_t build_queue, void* workspace, size_t workspace_bytes,
                              void* stream);

/*
 * The same step with an explicit choice of launches: `stages` is a bit set of pkv_stage.
 * pkv_decode(build_queue) == pkv_decode_stages(DECODE | MERGE | (build_queue ? BUILD : 0)).
 * A stage left out is simply not launched (the queue / the partial states of an earlier call in
 * `workspace` are used as they are): this is how bench.py times the decode kernel alone with CUDA
 * events and how a caller overlaps the builder of step t+1 with other work.  With MERGE left out
 * and more than one split per row, `out` is not written for those rows.
 */
typedef enum { PKV_STAGE_BUILD = 1, PKV_STAGE_DECODE = 2, PKV_STAGE_MERGE = 4, PKV_STAGE_ALL = 7 } pkv_stage;
PKV_API pkv_status pkv_decode_stages(const pkv_shape* shape, const pkv_split_policy* policy, const void* q,
                                     const void* k_cache, const void* v_cache, const int32_t* block_table,
                                     const int32_t* seq_lens, void* out, float* lse, float scale,
                                     uint32_t stages, void* workspace, size_t workspace_bytes, void* stream);

/*
 * Allocation-free entry point: pkv_decode(build_queue = 1) for callers that cannot provide device
 * scratch memory (code under CUDA graph capture, serving loops and harnesses that forbid
 * cudaMalloc).  The step's scratch -- queue header and counters, split_offsets, task list and the
 * split-local partial states (m, l, acc) of PAPER.md:56 and 71-75 -- lives in ONE static array of
 * PKV_STATIC_WORKSPACE_BYTES in the library's device image; every GPU that loads the library holds
 * those bytes until the process exits.  The caller passes inputs and outputs only (device pointers,
 * same meaning, layout and ownership as for pkv_decode).  The call makes no cudaMalloc / cudaFree and
 * calls no allocating library routine; it launches one small clear kernel (the layout's
 * pkv_workspace_init_bytes must start at zero and the array keeps the previous call's contents)
 * and then the launches of pkv_decode.
 *   - PKV_ERR_WORKSPACE, before any CUDA call, if pkv_workspace_bytes(shape, policy) exceeds
 *     PKV_STATIC_WORKSPACE_BYTES (pkv_last_error() states both numbers).  8 MiB holds about 500
 *     (row, split) pairs at Hkv = 8, G = 4, d = 128: B = 1 at any split count, B = 8 up to S = 32;
 *     BALANCED / AUTO policies size for 256 splits per row and fit only B = 1.
 *   - All calls on one device share the array: calls that OVERLAP on the GPU (two streams) race on
 *     it and give undefined results -- serialise them or use pkv_decode with workspaces of your own.
 *   - The array's address is looked up once per device (cudaGetSymbolAddress, with the calling
 *     thread's current device) on the first call on that device; make that first call outside
 *     stream capture.  pkv_get_counters / pkv_read_workqueue have no static variant.
 * Other errors as pkv_decode.
 */
#define PKV_STATIC_WORKSPACE_BYTES (8u << 20)
PKV_API size_t pkv_static_workspace_bytes(void);   /* = PKV_STATIC_WORKSPACE_BYTES of the loaded library */
PKV_API pkv_status pkv_decode_static(const pkv_shape* shape, const pkv_split_policy* policy, const void* q,
                                     const void* k_cache, const void* v_cache, const int32_t* block_table,
                                     const int32_t* seq_lens, void* out, float* lse, float scale, void* stream);

/*
 * Indexed rows ("Indexed Q/O. The extension can read Q rows and write output rows by
 * index, avoiding per-bucket index_select and index_copy_"): one decode step over a SUBSET of the
 * batch's rows, in place.  shape->B = number of launch rows; launch row i works on request row
 * row_index[i] (dev int32 [B], values in [0, rows of the caller's arrays)) of q, out, lse,
 * block_table AND seq_lens -- nothing is gathered or scattered by the caller.  The queue in the
 * workspace is in launch rows (pkv_task.row = i).  At most 512 rows per call.  Otherwise as
 * pkv_decode with build_queue = 1.  The workspace layout depends on shape->B: keep one workspace per
 * subset size (or zero its init bytes again when B changes); pkv_decode_buckets lays every bucket
 * out for the whole batch and has no such restriction.
 */
PKV_API pkv_status pkv_decode_indexed(const pkv_shape* shape, const pkv_split_policy* policy, const void* q,
                                      const void* k_cache, const void* v_cache, const int32_t* block_table,
                                      const int32_t* seq_lens, const int32_t* row_index, void* out, float* lse,
                                      float scale, void* workspace, size_t workspace_bytes, void* stream);

/*
 * Fused KV-append (+RoPE) before decode ("fused RoPE/KV-cache writes", future work there;
 * DESIGN.md reading A29).  seq_lens[i] = N_i already counts the new token; its position is N_i - 1.
 * In ONE decode launch: q is rotated to that position in registers (q itself is not modified); the
 * task that owns token N_i - 1 takes that token's K (rotated) and V from k_new / v_new instead of the
 * pool -- patched into its shared-memory stage, so there is no write -> read dependency through the
 * cache -- and writes both to the pool slot of token N_i - 1 (page block_table[i][(N_i-1)/P]) for
 * later steps.  k_cache / v_cache are therefore WRITTEN by this call.  Rows with N_i = 0 append nothing.
 *   k_new, v_new   dev [rows, Hkv, d] f16, indexed like q (by request row)
 *   rope_cos/_sin  dev float [rope_positions, d/2]: cos / sin of position * theta_c, rotate-half
 *                  pairing (channel c < d/2 with c + d/2); both NULL = no rotation.  The rotation is
 *                  evaluated in FP32 product by product (no FMA) and rounded to FP16, so the bytes in
 *                  the pool are reproducible by a plain CPU restatement.
 * One-byte caches (shape->kv_dtype E4M3 or INT8; reading A30): k_new / v_new stay FP16; the
 * (rotated) token is divided by its KV head's k_scale / v_scale in FP32 and rounded once to the cache's
 * code -- E4M3: to nearest even, magnitudes beyond 448 saturate; INT8: half to even, clamped to
 * [-127, 127] -- and that byte is what the pool receives and what this step attends over.
 * TMA kernel and d = 128 only (else PKV_ERR_UNSUPPORTED).  Otherwise as pkv_decode with
 * build_queue = 1; row_index may be NULL.
 */
typedef struct {
    const void* k_new;
    const void* v_new;
    const float* rope_cos;
    const float* rope_sin;
    int32_t rope_positions; /* rows of the tables; positions >= this are not rotated */
    int32_t reserved_;
} pkv_append;
PKV_API pkv_status pkv_decode_append(const pkv_shape* shape, const pkv_split_policy* policy, const void* q,
                                     void* k_cache, void* v_cache, const int32_t* block_table,
                                     const int32_t* seq_lens, const int32_t* row_index, const pkv_append* append,
                                     void* out, float* lse, float scale, void* workspace,
                                     size_t workspace_bytes, void* stream);

/*
 * Length-bucket route ("one per route length"; DESIGN.md readings
 * A22, A23) -- the route the compact workqueue replaces, kept as its comparator (Table 4: 16.00 vs
 * 2.00 launches per step).
 * pkv_plan_buckets_host (pure CPU): a row's route length is its true length rounded up to
 * bucket_tokens (1 = exact length buckets); rows of equal route length form a bucket; buckets in
 * ascending route length, rows ascending inside; rows with N_i <= 0 belong to no bucket and are
 * listed after the last one.  Writes row_index_out [B] (a permutation of 0..B-1),
 * bucket_offsets_out [B+1] (first num_buckets+1 entries used), bucket_lengths_out [B] or NULL.
 * pkv_decode_buckets: one pkv_decode_indexed per bucket over row_index[offsets[b] .. offsets[b+1])
 * (dev copy of the plan's row_index; bucket_offsets on the HOST), i.e. one decode (+ merge) launch
 * per bucket with the policy's route and split count, all on one workspace sized for the whole
 * batch; then one more launch for the rows of no bucket (out = 0, lse = -inf).
 * pkv_bucket_counters_host (pure CPU): Table 4's counters for that step, summed over the buckets
 * (policy.num_splits == 0 needs policy.num_sms > 0).
 */
PKV_API pkv_status pkv_plan_buckets_host(const int32_t* seq_lens_host, int32_t B, int32_t bucket_tokens,
                                         int32_t* row_index_out, int32_t* bucket_offsets_out,
                                         int32_t* bucket_lengths_out, int32_t* num_buckets_out);
PKV_API pkv_status pkv_decode_buckets(const pkv_shape* shape, const pkv_split_policy* policy, const void* q,
                                      const void* k_cache, const void* v_cache, const int32_t* block_table,
                                      const int32_t* seq_lens, const int32_t* row_index,
                                      const int32_t* bucket_offsets_host, int32_t num_buckets, void* out,
                                      float* lse, float scale, void* workspace, size_t workspace_bytes,
                                      void* stream);
PKV_API pkv_status pkv_bucket_counters_host(const pkv_shape* shape, const pkv_split_policy* policy,
                                            const int32_t* seq_lens_host, int32_t bucket_tokens,
                                            pkv_counters* out);

/*
 * Exact merge of split states (segmented over each row's compact slot range,
 * PAPER.md:75).  Public partial-state format, all FP32, natural-log domain:
 *   part_m [slots, G], part_l [slots, G], part_acc [slots, G, d],
 *   slot(i, g, s) = split_offsets[i]*Hkv + g*n_i + s,  n_i = split_offsets[i+1]-split_offsets[i]
 * Neutral states (m = -inf, l = 0) drop out; a row with no state or only neutral states gives
 * out = 0, lse = -inf.  split_offsets is dev [B+1].
 */
PKV_API pkv_status pkv_merge(const pkv_shape* shape, const float* part_m, const float* part_l,
                             const float* part_acc, const int32_t* split_offsets, void* out,
                             float* lse, void* stream);

/* Host copies of the workspace's counters / queue.  These two SYNCHRONISE `stream`. */
PKV_API pkv_status pkv_get_counters(const pkv_shape* shape, const pkv_split_policy* policy,
                                    const void* workspace, size_t workspace_bytes,
                                    pkv_counters* host_out, void* stream);
PKV_API pkv_status pkv_read_workqueue(const pkv_shape* shape, const pkv_split_policy* policy,
                                      const void* workspace, size_t workspace_bytes,
                                      pkv_task* host_tasks, int32_t cap, int32_t* host_split_offsets,
                                      int32_t* host_num_tasks, void* stream);
/* Test hook: device pointers of the partial states inside the workspace (no sync). */
PKV_API pkv_status pkv_workspace_partials(const pkv_shape* shape, const pkv_split_policy* policy,
                                          void* workspace, size_t workspace_bytes, float** part_m,
                                          float** part_l, float** part_acc, int64_t* slots_cap);

/*
 * One decode step with HOST buffers (the serving-facing path of PAPER.md:122-126: per-step
 * metadata is planned on the host and uploaded; bench.py's e2e leg).  The K/V page pool is the
 * model's resident state and stays on the device; q, block_table and seq_lens come from the
 * host, out goes back to the host.  The call
 *   1. plans on the host from seq_lens_host -- with PKV_SPLIT_AUTO the cost model first picks the
 *      step's policy -- but only the COUNTS of the queue (tasks, max_i n_i, (row, split) pairs):
 *      they decide which launches happen, so decode/merge launch counts equal the oracle's
 *      (A13); the queue itself is derived from the uploaded lengths inside the decode
 *      kernel (fused build) and is bit-identical to pkv_build_workqueue_host's,
 *   2. copies seq_lens and q to `dev_scratch` with ONE cudaMemcpyAsync, and of the block table only
 *      the rows whose used entries changed since the previous call on the same (host_staging,
 *      dev_scratch) pair -- `host_staging` keeps the shadow; a growing row changes one entry every
 *      page_size steps, so most steps upload no table bytes at all,
 *   3. launches decode (+ merge), and
 *   4. gets out to out_host -- when out_host is pinned, device-mapped memory a small kernel chained
 *      behind the merge stores it there (no copy-engine hop), else one cudaMemcpyAsync -- and
 *      SYNCHRONISES the stream.
 * host_staging: host memory of pkv_host_scratch_bytes() bytes (pinned recommended), zeroed (or
 * never used with another dev_scratch) before its first use; dev_scratch: device memory of the same
 * size, 256-byte aligned; the pair must be passed together from step to step.  counters_out may be
 * NULL.
 */
PKV_API size_t pkv_host_scratch_bytes(const pkv_shape* shape, const pkv_split_policy* policy);
PKV_API pkv_status pkv_decode_host(const pkv_shape* shape, const pkv_split_policy* policy,
                                   const void* q_host, const void* k_cache_dev, const void* v_cache_dev,
                                   const int32_t* block_table_host, const int32_t* seq_lens_host,
                                   void* out_host, float scale, void* host_staging, void* dev_scratch,
                                   size_t scratch_bytes, void* workspace, size_t workspace_bytes,
                                   void* stream, pkv_counters* counters_out);

/*
 * The host-buffer step with its submission taken off the critical path (the serving-
 * facing time includes planning and launching).  A synchronous step pays, before its first kernel
 * runs, the driver calls that enqueue it and the start of a kernel on an idle GPU, and after its last
 * the wake-up of the synchronising thread -- about 20 us of a 45 us config-2 step.  Here the caller
 * tells the call what the NEXT step will be (`next`: its lengths and block table -- a decode loop knows
 * them when it schedules: N + 1 for every continuing row -- and optionally other caches / another
 * out_host).  While the GPU works on this step, the call plans the next one, writes its lengths and
 * changed table rows into the staging image and enqueues its launches BEHIND A GATE:
 *       gate / stage kernel -> decode -> merge -> signal kernel
 * The gate is one CTA that polls a flag word of the pinned staging buffer over the host link; once the
 * host has released the step it fetches lengths, q and table rows from the image into dev_scratch.
 * Decode, merge and signal are chained behind it by programmatic launch: they are resident and
 * planned when the gate opens.  Decode and merge write the result into dev_scratch; the signal kernel
 * copies it into the pinned out_host and writes the step's number into a done word of the image.  The
 * next call then only copies q into the image, stores the flag (before it validates or plans anything,
 * when it repeats the armed step's arguments byte for byte) and spins on the done word.
 * Results are those of pkv_decode_host, bit for bit (the same kernels on the same inputs).
 *   - Needs: host_staging and out_host pinned and device-mapped, host_staging 256-byte aligned, the TMA
 *     kernel with the fused build (B <= 512), no PKV_FLAG_VALIDATE / SEPARATE_BUILD, at most 256 KiB of
 *     inputs in at most four pieces per step.  Otherwise -- and whenever the armed step turns out not to
 *     be the one the next call asks for (other lengths, table, buffers, policy) -- the call does what
 *     pkv_decode_host does; a mispredicted armed step is first run on whatever the image holds and its
 *     result discarded.  A step is only armed when the kernels it launches have run before in this
 *     thread.
 *   - WHILE A STEP IS ARMED THE STREAM IS BLOCKED by the polling gate: anything that waits for the stream
 *     or for the whole device (cudaStreamSynchronize, cudaDeviceSynchronize, cudaFree, cudaMemcpy)
 *     does not return until the step is released -- or until the gate gives up, 200 ms after it
 *     started; such an expired step runs on stale inputs, is marked, and the next call redoes it.
 *     pkv_decode_host_drain(host_staging, stream) releases an armed step at once (it runs on stale
 *     inputs; its result is discarded) and waits for it.  pkv_decode_host drains its staging buffer
 *     itself.  State is per (thread, host_staging): call from one thread.
 *   - next == NULL (or next->seq_lens_host == NULL): nothing is armed; the call is a synchronous step
 *     that waits on the done word instead of cudaStreamSynchronize.
 * Arguments as pkv_decode_host.
 */
typedef struct {
    const int32_t* seq_lens_host;    /* [B] the next step's lengths                                     */
    const int32_t* block_table_host; /* [B, max_pages] the next step's table                            */
    const void* k_cache_dev;         /* NULL = the same caches as this step                              */
    const void* v_cache_dev;
    void* out_host;                  /* NULL = the same out_host                                         */
} pkv_next_step;
PKV_API pkv_status pkv_decode_host_pipelined(const pkv_shape* shape, const pkv_split_policy* policy,
                                             const void* q_host, const void* k_cache_dev, const void* v_cache_dev,
                                             const int32_t* block_table_host, const int32_t* seq_lens_host,
                                             void* out_host, float scale, void* host_staging, void* dev_scratch,
                                             size_t scratch_bytes, void* workspace, size_t workspace_bytes,
                                             void* stream, const pkv_next_step* next, pkv_counters* counters_out);
PKV_API pkv_status pkv_decode_host_drain(void* host_staging, void* stream);

/*
 * The calibrated cost model (sec. 3.5), on the HOST, from host-resident lengths --
 * as the paper's harness evaluates it before every decode step:
 *     T_r = KVBytes / beta * max(1, C_min / C_r) + L_r * lambda + MergeBytes_r / beta
 * KVBytes = sum_i N_i * 2*Hkv*d*2, C_r = tasks / num_sms (Table 4's "Decode CTA work/SM"), L_r =
 * decode + merge launches, MergeBytes_r as pkv_counters.merge_bytes (0 when no row has two slots).
 * bucket_tokens > 0 evaluates the length-bucket route (totals over the buckets, A23),
 * 0 the policy's single launch pair.  `makespan_us` is the B200 re-fit of the first term (DESIGN.md
 * A27): max(KVBytes/beta, busiest CTA's bytes / beta_cta), beta_cta = beta / (C_min * num_sms) --
 * equal to the paper's term when all tasks are equal, larger when one share dominates.
 * pkv_default_cost_model: the constants fitted on B200 this round;
 * pkv_calibrate measures beta and lambda on the device at hand.
 * pkv_choose_policy: evaluates the library's candidate policies for this step -- BALANCED, and
 * FIXED_COUNT with S in {1, 2, 4, ..., 128} on 32-token tiles, all on `base`'s route, merge mode,
 * kernel and flags -- and writes the winner to `chosen`: among the candidates whose makespan_total_us
 * is within 1 % of the smallest, the one whose units cover the most SMs (min(units, num_sms); the
 * model cannot tell such candidates apart, and measured steps favour the fuller machine: config 2,
 * 147 vs 128 units: 23.4 vs 23.8 us), then the smaller estimate, then FIXED_COUNT before BALANCED (the
 * same decomposition with the shorter in-kernel plan) and the smaller S.
 * PKV_SPLIT_AUTO in pkv_decode_host does this per step.
 */
typedef struct {
    double beta_gbps;  /* streaming read bandwidth                                   (paper: 331.2) */
    double lambda_us;  /* cost of one more dependent kernel launch in a decode step  (paper: 8.19)  */
    double c_min;      /* work items per SM that saturate beta                       (paper: 4)     */
    int32_t num_sms;   /*                                                            (paper: 28)    */
    int32_t reserved_;
} pkv_cost_model;
typedef struct {
    double total_us, stream_us, launch_us, merge_us; /* the paper's formula, term by term            */
    double cta_work_per_sm;                          /* C_r                                          */
    double makespan_us, makespan_total_us;           /* A27: first term, and the total with it        */
    int64_t kv_bytes, merge_bytes, tasks, launches, max_share_bytes;
    int64_t units;                                   /* CTA work units of the launch(es): (row, split) pairs x head groups */
} pkv_cost_estimate;
PKV_API pkv_status pkv_default_cost_model(int32_t num_sms, pkv_cost_model* out);
PKV_API pkv_status pkv_estimate_cost(const pkv_shape* shape, const pkv_split_policy* policy,
                                     const int32_t* seq_lens_host, int32_t bucket_tokens,
                                     const pkv_cost_model* model, pkv_cost_estimate* out);
PKV_API pkv_status pkv_choose_policy(const pkv_shape* shape, const int32_t* seq_lens_host,
                                     const pkv_cost_model* model, const pkv_split_policy* base,
                                     pkv_split_policy* chosen, pkv_cost_estimate* estimate_out);

/*
 * Calibration of the paper's cost-model constants on the current device ("beta is
 * measured streaming read bandwidth ... lambda is a calibrated launch-overhead constant ... a
 * different GPU should re-fit them").  dev_buffer: device memory, 256-byte aligned, at least 64 MiB
 * (use several times the L2 size: it is read end to end, its first word may be written).  Runs
 * probe kernels on a stream of its own after synchronising `stream`; allocates two events, a
 * stream and a graph; NOT capture-safe; takes tens of milliseconds.
 */
typedef struct {
    double read_gbps;           /* beta: the best of the three read probes below, GB/s                 */
    double read_ldg_gbps;       /* 16-byte ld.global.nc loads, persistent grid of 4 CTAs per SM        */
    double read_bulk8k_gbps;    /* cp.async.bulk 8 KiB chunks into a 12-stage shared-memory ring, 1 CTA/SM */
    double read_bulk16k_gbps;   /* the same with 16 KiB chunks                                         */
    double launch_us;           /* lambda: per kernel of a chain of empty kernels launched into a stream */
    double launch_pdl_us;       /* the same with programmatic dependent launch                         */
    double graph_launch_us;     /* the same chain replayed from a CUDA graph                           */
    double graph_launch_pdl_us; /* graph + programmatic dependent launch (what a decode step pays)     */
    int64_t buffer_bytes;
    int32_t num_sms, l2_bytes;
} pkv_calibration;
PKV_API pkv_status pkv_calibrate(void* dev_buffer, size_t bytes, void* stream, pkv_calibration* out);

#ifdef __cplusplus
}
#endif
#endif /* PKV_H_ */
