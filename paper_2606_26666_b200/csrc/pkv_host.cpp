// pkv_host.cpp -- the pure-CPU part of libpkv: argument validation, policy resolution,
// workspace layout and the host workqueue planner.  No CUDA here.
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <algorithm>
#include <utility>
#include <vector>

#include "pkv_common.h"

namespace pkv {

static thread_local char g_error[512] = "";

void set_error(const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_error, sizeof(g_error), fmt, ap);
    va_end(ap);
}
void clear_error() { g_error[0] = 0; }

pkv_status validate_and_resolve(const pkv_shape* shape, const pkv_split_policy* policy,
                                int num_sms_or_0, bool bound_ok, Resolved* out) {
    if (!shape || !policy || !out) { set_error("null shape/policy"); return PKV_ERR_INVALID_ARG; }
    const pkv_shape& s = *shape;
    const pkv_split_policy& p = *policy;
    if (s.B < 0 || s.Hq <= 0 || s.Hkv <= 0 || s.d <= 0 || s.page_size <= 0 || s.max_pages < 0 ||
        s.num_pages < 0) {
        set_error("negative or zero dimension in pkv_shape");
        return PKV_ERR_INVALID_ARG;
    }
    if (s.Hq % s.Hkv != 0) { set_error("Hq=%d is not a multiple of Hkv=%d", s.Hq, s.Hkv); return PKV_ERR_INVALID_ARG; }
    if (s.d != 64 && s.d != 128 && s.d != 256) { set_error("d=%d not compiled in (64, 128 or 256)", s.d); return PKV_ERR_UNSUPPORTED; }
    if (s.page_size != 16 && s.page_size != 32 && s.page_size != 64) { set_error("page_size=%d not supported (16, 32 or 64)", s.page_size); return PKV_ERR_UNSUPPORTED; }
    const int G = s.Hq / s.Hkv;
    if (G != 1 && G != 2 && G != 4 && G != 8 && G != 16) { set_error("G=Hq/Hkv=%d not compiled in (1, 2, 4, 8 and 16 only)", G); return PKV_ERR_UNSUPPORTED; }
    if (s.kv_dtype != PKV_KV_F16 && s.kv_dtype != PKV_KV_E4M3 && s.kv_dtype != PKV_KV_INT8) { set_error("bad kv_dtype %d", s.kv_dtype); return PKV_ERR_INVALID_ARG; }
    if (s.kv_dtype != PKV_KV_F16) {
        if (s.d != kD) { set_error("one-byte KV caches are compiled in for d=128 only (d=%d)", s.d); return PKV_ERR_UNSUPPORTED; }
        if (p.kernel == PKV_KERNEL_SIMT) { set_error("FP8 KV needs the TMA kernel"); return PKV_ERR_UNSUPPORTED; }
        if (s.kv_stride_page % 16 || s.kv_stride_token % 16 || s.kv_stride_head % 16) { set_error("FP8 kv strides must be multiples of 16 bytes"); return PKV_ERR_INVALID_ARG; }
    }
    const bool default_strides = s.kv_stride_page == 0 && s.kv_stride_token == 0 && s.kv_stride_head == 0;
    if (!default_strides) {
        if (s.kv_stride_page <= 0 || s.kv_stride_token <= 0 || s.kv_stride_head <= 0) {
            set_error("kv strides must be all zero (default layout) or all positive");
            return PKV_ERR_INVALID_ARG;
        }
        if (s.kv_stride_page % 8 || s.kv_stride_token % 8 || s.kv_stride_head % 8) {
            set_error("kv strides must be multiples of 8 elements (16 bytes)");
            return PKV_ERR_INVALID_ARG;
        }
    }
    if (p.tile_tokens <= 0 || p.tile_tokens % s.page_size != 0) {
        set_error("tile_tokens=%d must be a positive multiple of page_size=%d", p.tile_tokens, s.page_size);
        return PKV_ERR_INVALID_ARG;
    }
    if (p.split_mode != PKV_SPLIT_FIXED_COUNT && p.split_mode != PKV_SPLIT_FIXED_CHUNK &&
        p.split_mode != PKV_SPLIT_BALANCED && p.split_mode != PKV_SPLIT_AUTO) {
        set_error("bad split_mode %d", p.split_mode);
        return PKV_ERR_INVALID_ARG;
    }
    if (p.num_splits < 0 || p.num_splits > kMaxSplits) {
        set_error("num_splits=%d outside [0, %d]", p.num_splits, kMaxSplits);
        return PKV_ERR_INVALID_ARG;
    }
    if (p.split_mode == PKV_SPLIT_FIXED_CHUNK && p.chunk_tiles <= 0) {
        set_error("FIXED_CHUNK needs chunk_tiles > 0");
        return PKV_ERR_INVALID_ARG;
    }
    if (p.route != PKV_ROUTE_RECT && p.route != PKV_ROUTE_WORKQUEUE) { set_error("bad route %d", p.route); return PKV_ERR_INVALID_ARG; }
    if (p.merge_mode != PKV_MERGE_SEPARATE && p.merge_mode != PKV_MERGE_FUSED) { set_error("bad merge_mode %d", p.merge_mode); return PKV_ERR_INVALID_ARG; }
    if (p.kernel < PKV_KERNEL_AUTO || p.kernel > PKV_KERNEL_SIMT) { set_error("bad kernel %d", p.kernel); return PKV_ERR_INVALID_ARG; }
    if (p.num_sms < 0) { set_error("num_sms < 0"); return PKV_ERR_INVALID_ARG; }
    if (p.flags & ~(int32_t)kAllFlags) { set_error("unknown policy flag bits 0x%x", p.flags); return PKV_ERR_INVALID_ARG; }
    if (p.heads_per_cta != 0 && ((p.heads_per_cta != 1 && p.heads_per_cta != 2 && p.heads_per_cta != 4 && p.heads_per_cta != 8) ||
                                 s.Hkv % p.heads_per_cta != 0)) {
        set_error("heads_per_cta=%d must be 0 (auto), 1, 2, 4 or 8 and divide Hkv=%d", p.heads_per_cta, s.Hkv);
        return PKV_ERR_INVALID_ARG;
    }
    if (p.heads_per_cta > max_heads_per_cta(G, s.d)) { set_error("heads_per_cta=8 is not available with G=16 or d=256 (at most 4)"); return PKV_ERR_INVALID_ARG; }
    if (s.d != kD && p.kernel == PKV_KERNEL_SIMT) { set_error("PKV_KERNEL_SIMT is compiled in for d=128 only"); return PKV_ERR_UNSUPPORTED; }

    int32_t S = p.num_splits;
    out->num_sms = p.num_sms > 0 ? p.num_sms : num_sms_or_0;
    const bool balanced = p.split_mode == PKV_SPLIT_BALANCED || p.split_mode == PKV_SPLIT_AUTO;
    if (balanced && out->num_sms <= 0 && !bound_ok) {
        set_error("BALANCED needs policy.num_sms > 0 in a host-only call");
        return PKV_ERR_INVALID_ARG;
    }
    if (S == 0) {
        if (p.split_mode != PKV_SPLIT_FIXED_COUNT) {
            S = kMaxSplits;
        } else {
            int sms = p.num_sms > 0 ? p.num_sms : num_sms_or_0;
            if (sms > 0) {
                int64_t units = (int64_t)(s.B > 0 ? s.B : 1) * s.Hkv;
                int64_t want = ceil_div64((int64_t)kAutoCMin * sms, units);
                S = (int32_t)(want < 1 ? 1 : (want > kMaxSplits ? kMaxSplits : want));
            } else if (bound_ok) {
                S = kMaxSplits;
            } else {
                set_error("num_splits == 0 (auto) needs policy.num_sms > 0 in a host-only call");
                return PKV_ERR_INVALID_ARG;
            }
        }
    }
    out->S = S;
    out->tile_tokens = p.tile_tokens;
    out->split_mode = balanced ? (int32_t)PKV_SPLIT_BALANCED : p.split_mode;
    out->auto_mode = p.split_mode == PKV_SPLIT_AUTO ? 1 : 0;
    out->chunk_tiles = p.chunk_tiles > 0 ? p.chunk_tiles : 1;
    out->route = p.route;
    out->merge_mode = p.merge_mode;
    out->kernel = p.kernel == PKV_KERNEL_AUTO ? PKV_KERNEL_TMA_MMA : p.kernel;
    out->G = G;
    out->flags = p.flags;
    out->heads_per_cta = p.heads_per_cta;
    // default: 256 KiB of FP16 K/V per CTA (FP8: 128 KiB -- the same tokens); measured sweeps in DESIGN.md
    out->prefetch_kb = p.prefetch_kb == 0 ? (s.kv_dtype != PKV_KV_F16 ? kDefaultPrefetchKb / 2 : kDefaultPrefetchKb)
                                          : (p.prefetch_kb < 0 ? 0 : p.prefetch_kb);
    return PKV_OK;
}

WorkspaceLayout workspace_layout(const pkv_shape& s, int32_t S) {
    WorkspaceLayout L;
    const int G = s.Hq / s.Hkv;
    L.slots_cap = (int64_t)s.B * s.Hkv * S;
    size_t off = 0;
    L.header = off;         off = align_up(off + sizeof(QueueHeader), 256);
    L.fuse_counters = off;  off = align_up(off + sizeof(int32_t) * ((size_t)s.B * s.Hkv + 1), 256);
    L.init_bytes = off;     // header + completion counters: zero on first use (include/pkv.h)
    L.split_offsets = off;  off = align_up(off + sizeof(int32_t) * ((size_t)s.B + 1), 256);
    L.rowslots = off;       off = align_up(off + sizeof(RowSlot) * (size_t)s.B * S, 256);
    L.tasks = off;          off = align_up(off + sizeof(pkv_task) * (size_t)L.slots_cap, 256);
    L.part_m = off;         off = align_up(off + sizeof(float) * (size_t)L.slots_cap * G, 256);
    L.part_l = off;         off = align_up(off + sizeof(float) * (size_t)L.slots_cap * G, 256);
    L.part_acc = off;       off = align_up(off + sizeof(float) * (size_t)L.slots_cap * G * s.d, 256);
    L.total = off;
    return L;
}

pkv_status plan_host(const pkv_shape& s, const Resolved& rp, const int32_t* seq_lens, pkv_task* tasks,
                     int32_t tasks_cap, int32_t* split_offsets, RowSlot* rowslots, QueueHeader* hdr,
                     int32_t* max_unit_tokens) {
    int64_t count = 0, sum_seq = 0;
    int32_t max_tok = 0;
    int32_t max_n = 0, empties = 0, off = 0;
    bool overflow = false;
    int32_t chunk = rp.split_mode == PKV_SPLIT_FIXED_COUNT ? 0 : rp.chunk_tiles;
    if (rp.split_mode == PKV_SPLIT_BALANCED) {
        int64_t W = 0;
        for (int32_t i = 0; i < s.B; ++i)
            if (seq_lens[i] > 0) W += ((int64_t)seq_lens[i] + rp.tile_tokens - 1) / rp.tile_tokens;
        chunk = balanced_chunk(W, rp.num_sms, rp.tile_tokens, [&](int32_t c) {
            int64_t units = 0;
            for (int32_t i = 0; i < s.B; ++i)
                if (seq_lens[i] > 0) units += ((int64_t)seq_lens[i] + (int64_t)rp.tile_tokens * c - 1) / ((int64_t)rp.tile_tokens * c);
            return units <= rp.num_sms;
        });
    }
    if (split_offsets) split_offsets[0] = 0;
    for (int32_t i = 0; i < s.B; ++i) {
        const int32_t N = seq_lens[i] > 0 ? seq_lens[i] : 0;
        sum_seq += N;
        const RowSplits r = row_splits(N, rp.tile_tokens, rp.split_mode, rp.S, chunk);
        const int32_t slots = rp.route == PKV_ROUTE_WORKQUEUE ? r.n : rp.S;
        if (slots > max_n) max_n = slots;
        if (r.T > 0) {   // the row's largest token range: its first split (ceil-chunks, A6)
            const int64_t t1 = (int64_t)r.c * rp.tile_tokens;
            const int32_t tok = (int32_t)(t1 < N ? t1 : N);
            if (tok > max_tok) max_tok = tok;
        }
        if (!tasks) {   // counts only: no need to walk the row's tasks
            count += (int64_t)s.Hkv * slots;
            empties += (slots - r.n) * s.Hkv;
            if (tasks_cap == 0 && (int64_t)s.Hkv * slots > 0) overflow = true;
        }
        for (int32_t g = 0; tasks && g < s.Hkv; ++g) {
            for (int32_t sp = 0; sp < slots; ++sp) {
                int32_t tb = 0, te = 0;
                if (r.T > 0) {
                    int64_t b = (int64_t)sp * r.c, e = (int64_t)(sp + 1) * r.c;
                    tb = (int32_t)(b < r.T ? b : r.T);
                    te = (int32_t)(e < r.T ? e : r.T);
                }
                if (tb >= te) ++empties;
                if (count < tasks_cap && tasks) {
                    pkv_task t = {i, g, sp, tb, te};
                    tasks[count] = t;
                } else {
                    overflow = true;
                }
                ++count;
            }
        }
        if (rowslots) {
            for (int32_t sp = 0; sp < slots; ++sp) {
                RowSlot rs;
                std::memset(&rs, 0, sizeof(rs));
                rs.row = i; rs.so = off; rs.n = slots; rs.split = sp; rs.grow = i; rs.nlen = N;
                if (r.T > 0) {
                    const int64_t b = (int64_t)sp * r.c, e = (int64_t)(sp + 1) * r.c;
                    const int64_t t0 = (b < r.T ? b : r.T) * rp.tile_tokens, t1 = (e < r.T ? e : r.T) * rp.tile_tokens;
                    rs.tok0 = (int32_t)t0;
                    rs.tok1 = (int32_t)(t1 < N ? t1 : N);
                }
                rowslots[off + sp] = rs;
            }
        }
        off += slots;
        if (split_offsets) split_offsets[i + 1] = off;
    }
    if (hdr) {
        std::memset(hdr, 0, sizeof(*hdr));
        hdr->num_tasks = (int32_t)count;
        hdr->max_row_splits = max_n;
        hdr->total_row_slots = off;
        hdr->resolved_splits = rp.S;
        hdr->empty_tasks = empties;
        hdr->sum_seq_lens = sum_seq;
        hdr->chunk_tiles = chunk;
    }
    if (max_unit_tokens) *max_unit_tokens = max_tok;
    if (overflow && tasks) return PKV_ERR_WORKSPACE;
    return PKV_OK;
}

namespace {

// Totals of one launch pair (policy resolved, lengths on the host) for the cost model.
struct RouteTotals {
    int64_t kv_bytes = 0, merge_bytes = 0, tasks = 0, launches = 0;
    int64_t max_share = 0, units = 0;
    double slice_eff = 1.0;   // A27: head_slice_efficiency of the launch's heads per CTA
};

void launch_totals(const pkv_shape& s, const Resolved& rp, const int32_t* lens, int num_sms, RouteTotals* t) {
    QueueHeader hdr;
    int32_t max_tok = 0;
    plan_host(s, rp, lens, nullptr, 0, nullptr, nullptr, &hdr, &max_tok);
    const bool partials = hdr.max_row_splits > 1;
    t->kv_bytes = hdr.sum_seq_lens * 2 * s.Hkv * s.d * (s.kv_dtype != PKV_KV_F16 ? 1 : 2);
    t->tasks = hdr.num_tasks;
    t->merge_bytes = partials ? (int64_t)hdr.num_tasks * rp.G * (s.d + 2) * 4 : 0;
    t->launches = (hdr.num_tasks > 0 ? 1 : 0) + ((partials && hdr.num_tasks > 0 && rp.merge_mode == PKV_MERGE_SEPARATE) ? 1 : 0);
    // A27: the busiest CTA's bytes.  A unit = the HG tasks of one (row, split) token range.
    t->max_share = 0;
    if (hdr.total_row_slots > 0) {
        const int hg = choose_heads_per_cta(rp.heads_per_cta, s.Hkv, hdr.total_row_slots, num_sms, max_heads_per_cta(rp.G, s.d));
        const int64_t unit = (int64_t)max_tok * 2 * hg * s.d * (s.kv_dtype != PKV_KV_F16 ? 1 : 2);
        const int64_t units = (int64_t)hdr.total_row_slots * (s.Hkv / hg);
        // several waves: units are handed out dynamically when every (head, block) group of a CTA is one
        // warp (HG x blocks = 8), else round-robin -- then the busiest CTA may draw only largest units
        const bool dynamic = hg * (rp.G == 16 ? 2 : 1) == 8;
        const int64_t waves = (units + num_sms - 1) / num_sms;
        t->max_share = units <= num_sms ? unit : (dynamic ? t->kv_bytes / num_sms + unit : waves * unit);
        t->units = units;
        t->slice_eff = head_slice_efficiency(hg);
    }
}

}  // namespace

}  // namespace pkv

using namespace pkv;

extern "C" {

int32_t pkv_version(void) { return (2 << 16) | 0; }
const char* pkv_last_error(void) { return g_error; }

size_t pkv_workspace_bytes(const pkv_shape* shape, const pkv_split_policy* policy) {
    Resolved rp;
    if (validate_and_resolve(shape, policy, 0, /*bound_ok=*/true, &rp) != PKV_OK) return 0;
    return workspace_layout(*shape, rp.S).total;
}

size_t pkv_workspace_init_bytes(const pkv_shape* shape, const pkv_split_policy* policy) {
    Resolved rp;
    if (validate_and_resolve(shape, policy, 0, /*bound_ok=*/true, &rp) != PKV_OK) return 0;
    return workspace_layout(*shape, rp.S).init_bytes;
}

pkv_status pkv_plan_buckets_host(const int32_t* seq_lens_host, int32_t B, int32_t bucket_tokens, int32_t* row_index_out,
                                 int32_t* bucket_offsets_out, int32_t* bucket_lengths_out, int32_t* num_buckets_out) {
    clear_error();
    if (B < 0 || bucket_tokens <= 0 || !num_buckets_out || (B > 0 && (!seq_lens_host || !row_index_out || !bucket_offsets_out))) {
        set_error("pkv_plan_buckets_host: bad argument");
        return PKV_ERR_INVALID_ARG;
    }
    // route length = true length rounded up to the granularity; stable sort of the non-empty rows
    // by route length (ascending), empty rows last (reading A22)
    std::vector<std::pair<int64_t, int32_t>> keyed;
    keyed.reserve((size_t)B);
    for (int32_t i = 0; i < B; ++i)
        if (seq_lens_host[i] > 0)
            keyed.emplace_back(((int64_t)seq_lens_host[i] + bucket_tokens - 1) / bucket_tokens * bucket_tokens, i);
    std::stable_sort(keyed.begin(), keyed.end(),
                     [](const std::pair<int64_t, int32_t>& a, const std::pair<int64_t, int32_t>& b) { return a.first < b.first; });
    int32_t nb = 0, pos = 0;
    if (bucket_offsets_out) bucket_offsets_out[0] = 0;
    for (size_t k = 0; k < keyed.size(); ++k) {
        if (k > 0 && keyed[k].first != keyed[k - 1].first) bucket_offsets_out[++nb] = pos;
        if (bucket_lengths_out && (k == 0 || keyed[k].first != keyed[k - 1].first))
            bucket_lengths_out[k == 0 ? 0 : nb] = (int32_t)(keyed[k].first < 0x7fffffff ? keyed[k].first : 0x7fffffff);
        row_index_out[pos++] = keyed[k].second;
    }
    if (!keyed.empty()) bucket_offsets_out[++nb] = pos;
    for (int32_t i = 0; i < B; ++i)
        if (seq_lens_host[i] <= 0) row_index_out[pos++] = i;
    *num_buckets_out = nb;
    return PKV_OK;
}

pkv_status pkv_bucket_counters_host(const pkv_shape* shape, const pkv_split_policy* policy, const int32_t* seq_lens_host,
                                    int32_t bucket_tokens, pkv_counters* out) {
    clear_error();
    Resolved rp0;
    pkv_status st = validate_and_resolve(shape, policy, 0, /*bound_ok=*/false, &rp0);
    if (st != PKV_OK) return st;
    if (!out || (shape->B > 0 && !seq_lens_host) || bucket_tokens <= 0) { set_error("pkv_bucket_counters_host: bad argument"); return PKV_ERR_INVALID_ARG; }
    const int32_t B = shape->B;
    std::vector<int32_t> index((size_t)B), offs((size_t)B + 1), lens;
    int32_t nb = 0;
    st = pkv_plan_buckets_host(seq_lens_host, B, bucket_tokens, index.data(), offs.data(), nullptr, &nb);
    if (st != PKV_OK) return st;
    std::memset(out, 0, sizeof(*out));
    for (int32_t b = 0; b < nb; ++b) {
        pkv_shape sub = *shape;
        sub.B = offs[b + 1] - offs[b];
        Resolved rp;
        st = validate_and_resolve(&sub, policy, 0, false, &rp);   // the auto split count follows the bucket's size
        if (st != PKV_OK) return st;
        lens.assign((size_t)sub.B, 0);
        for (int32_t i = 0; i < sub.B; ++i) lens[i] = seq_lens_host[index[offs[b] + i]];
        QueueHeader hdr;
        plan_host(sub, rp, lens.data(), nullptr, 0, nullptr, nullptr, &hdr);
        const bool merge = hdr.max_row_splits > 1;
        out->tasks += hdr.num_tasks;
        out->empty_tasks += hdr.empty_tasks;
        out->decode_launches += hdr.num_tasks > 0 ? 1 : 0;
        out->merge_launches += (merge && rp.merge_mode == PKV_MERGE_SEPARATE) ? 1 : 0;
        out->useful_kv_bytes += hdr.sum_seq_lens * 2 * shape->Hkv * shape->d * (shape->kv_dtype != PKV_KV_F16 ? 1 : 2);
        out->merge_bytes += merge ? (int64_t)hdr.num_tasks * rp.G * (shape->d + 2) * 4 : 0;
        out->num_splits = rp.S;
        if (hdr.max_row_splits > out->max_row_splits) out->max_row_splits = hdr.max_row_splits;
    }
    return PKV_OK;
}

pkv_status pkv_default_cost_model(int32_t num_sms, pkv_cost_model* out) {
    clear_error();
    if (!out || num_sms <= 0) { set_error("pkv_default_cost_model: bad argument"); return PKV_ERR_INVALID_ARG; }
    out->beta_gbps = kB200BetaGbps;
    out->lambda_us = kB200LambdaUs;
    out->c_min = kB200CMin;
    out->num_sms = num_sms;
    out->reserved_ = 0;
    return PKV_OK;
}

pkv_status pkv_estimate_cost(const pkv_shape* shape, const pkv_split_policy* policy, const int32_t* seq_lens_host,
                             int32_t bucket_tokens, const pkv_cost_model* model, pkv_cost_estimate* out) {
    clear_error();
    if (!model || !out || model->beta_gbps <= 0.0 || model->c_min <= 0.0 || model->num_sms <= 0 || bucket_tokens < 0) {
        set_error("pkv_estimate_cost: bad model or argument");
        return PKV_ERR_INVALID_ARG;
    }
    pkv_split_policy pol;
    if (policy) pol = *policy;
    if (policy && pol.num_sms == 0) pol.num_sms = model->num_sms;   // auto rule and BALANCED follow the model's machine
    Resolved rp;
    pkv_status st = validate_and_resolve(shape, policy ? &pol : nullptr, 0, /*bound_ok=*/false, &rp);
    if (st != PKV_OK) return st;
    if (shape->B > 0 && !seq_lens_host) { set_error("null seq_lens"); return PKV_ERR_INVALID_ARG; }
    const double beta = model->beta_gbps * 1e3;                                  // bytes per microsecond
    const double beta_cta = model->beta_gbps / (model->c_min * model->num_sms) * 1e3;
    RouteTotals sum;
    double makespan = 0.0;
    if (bucket_tokens == 0) {
        launch_totals(*shape, rp, seq_lens_host, model->num_sms, &sum);
        const double a = (double)sum.kv_bytes / (beta * sum.slice_eff), b = (double)sum.max_share / beta_cta;
        makespan = a > b ? a : b;
    } else {
        const int32_t B = shape->B;
        std::vector<int32_t> index((size_t)B), offs((size_t)B + 1), lens;
        int32_t nb = 0;
        st = pkv_plan_buckets_host(seq_lens_host, B, bucket_tokens, index.data(), offs.data(), nullptr, &nb);
        if (st != PKV_OK) return st;
        for (int32_t b = 0; b < nb; ++b) {   // buckets run one after the other: their makespans add up
            pkv_shape sub = *shape;
            sub.B = offs[b + 1] - offs[b];
            Resolved rb;
            st = validate_and_resolve(&sub, &pol, 0, false, &rb);
            if (st != PKV_OK) return st;
            lens.assign((size_t)sub.B, 0);
            for (int32_t i = 0; i < sub.B; ++i) lens[i] = seq_lens_host[index[offs[b] + i]];
            RouteTotals t;
            launch_totals(sub, rb, lens.data(), model->num_sms, &t);
            sum.kv_bytes += t.kv_bytes; sum.merge_bytes += t.merge_bytes; sum.tasks += t.tasks; sum.launches += t.launches;
            sum.units += t.units;
            if (t.max_share > sum.max_share) sum.max_share = t.max_share;
            const double a = (double)t.kv_bytes / (beta * t.slice_eff), c = (double)t.max_share / beta_cta;
            makespan += a > c ? a : c;
        }
    }
    // PAPER.md:83, term by term
    const double c_r = (double)sum.tasks / (double)model->num_sms;
    const double occupancy = c_r > 0.0 ? (model->c_min / c_r > 1.0 ? model->c_min / c_r : 1.0) : 1.0;
    out->stream_us = (double)sum.kv_bytes / beta * occupancy;
    out->launch_us = (double)sum.launches * model->lambda_us;
    out->merge_us = (double)sum.merge_bytes / beta;
    out->total_us = out->stream_us + out->launch_us + out->merge_us;
    out->cta_work_per_sm = c_r;
    out->makespan_us = makespan;
    out->makespan_total_us = makespan + out->launch_us + out->merge_us;
    out->kv_bytes = sum.kv_bytes; out->merge_bytes = sum.merge_bytes; out->tasks = sum.tasks; out->launches = sum.launches;
    out->max_share_bytes = sum.max_share;
    out->units = sum.units;
    return PKV_OK;
}

pkv_status pkv_choose_policy(const pkv_shape* shape, const int32_t* seq_lens_host, const pkv_cost_model* model,
                             const pkv_split_policy* base, pkv_split_policy* chosen, pkv_cost_estimate* estimate_out) {
    clear_error();
    if (!base || !chosen || !model) { set_error("pkv_choose_policy: null argument"); return PKV_ERR_INVALID_ARG; }
    pkv_split_policy cand[10];
    pkv_cost_estimate est[10];
    int n = 0;
    // candidates: BALANCED on page-size tiles, then FIXED_COUNT S = 1, 2, 4, ..., 128 and the
    // single-wave fit S = floor(SMs / (B * head groups)) on 32-token tiles
    const int sms = base->num_sms > 0 ? base->num_sms : model->num_sms;
    int s_fit = 0;
    if (shape && shape->B > 0 && shape->Hkv > 0 && shape->Hq % shape->Hkv == 0) {
        const int mh = max_heads_per_cta(shape->Hq / shape->Hkv, shape->d);
        int hg = mh;
        while (hg > 1 && (hg > shape->Hkv || shape->Hkv % hg)) hg >>= 1;
        s_fit = sms / (shape->B * (shape->Hkv / hg));
        if (s_fit > kMaxSplits) s_fit = kMaxSplits;
    }
    for (int c = -1; c <= 8; ++c) {
        if (c == 8 && (s_fit < 2 || (s_fit & (s_fit - 1)) == 0)) continue;   // nothing new to try
        pkv_split_policy pol = *base;
        pol.num_sms = base->num_sms > 0 ? base->num_sms : model->num_sms;
        if (c < 0) {
            pol.split_mode = PKV_SPLIT_BALANCED;
            pol.tile_tokens = shape ? shape->page_size : 16;
            pol.num_splits = 0;
        } else {
            pol.split_mode = PKV_SPLIT_FIXED_COUNT;
            pol.tile_tokens = 32;
            pol.num_splits = c == 8 ? s_fit : 1 << c;
        }
        const pkv_status st = pkv_estimate_cost(shape, &pol, seq_lens_host, 0, model, &est[n]);
        if (st != PKV_OK) return st;
        cand[n++] = pol;
    }
    int lo = 0;
    for (int i = 1; i < n; ++i)
        if (est[i].makespan_total_us < est[lo].makespan_total_us) lo = i;
    auto coverage = [&](int i) { return est[i].units < sms ? est[i].units : (int64_t)sms; };
    int pick = lo;
    for (int i = 0; i < n; ++i) {
        if (est[i].makespan_total_us > 1.01 * est[lo].makespan_total_us) continue;
        // equal coverage and estimate (the same decomposition): FIXED_COUNT, whose in-kernel plan is
        // shorter than BALANCED's (config 2: 23.4 vs 23.8 us per step)
        const bool better_tie = coverage(i) == coverage(pick) && est[i].makespan_total_us == est[pick].makespan_total_us &&
                                cand[pick].split_mode == PKV_SPLIT_BALANCED && cand[i].split_mode == PKV_SPLIT_FIXED_COUNT;
        if (coverage(i) > coverage(pick) || (coverage(i) == coverage(pick) && est[i].makespan_total_us < est[pick].makespan_total_us) ||
            better_tie)
            pick = i;
    }
    pkv_split_policy best = cand[pick];
    const pkv_cost_estimate best_est = est[pick];
    best.num_sms = base->num_sms;   // 0 stays "the device's": the estimate assumed the model's machine
    *chosen = best;
    if (estimate_out) *estimate_out = best_est;
    return PKV_OK;
}

pkv_status pkv_build_workqueue_host(const pkv_shape* shape, const pkv_split_policy* policy,
                                    const int32_t* seq_lens_host, pkv_task* tasks_out, int32_t tasks_cap,
                                    int32_t* split_offsets_out, int32_t* num_tasks_out) {
    clear_error();
    Resolved rp;
    pkv_status st = validate_and_resolve(shape, policy, 0, /*bound_ok=*/false, &rp);
    if (st != PKV_OK) return st;
    if ((!seq_lens_host && shape->B > 0) || !num_tasks_out || tasks_cap < 0 || (tasks_cap > 0 && !tasks_out)) {
        set_error("null pointer in pkv_build_workqueue_host");
        return PKV_ERR_INVALID_ARG;
    }
    QueueHeader hdr;
    st = plan_host(*shape, rp, seq_lens_host, tasks_out, tasks_cap, split_offsets_out, nullptr, &hdr);
    *num_tasks_out = hdr.num_tasks;
    if (st == PKV_ERR_WORKSPACE) set_error("tasks_cap=%d < %d tasks", tasks_cap, hdr.num_tasks);
    return st;
}

}  // extern "C"
