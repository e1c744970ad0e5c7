// pkdg.cu -- host side of the C ABI declared in include/pkdg.h.  No CPU fallback exists: every
// entry point either runs the CUDA kernels of pkdg_kernels.cuh or returns an error.
#include "../../include/pkdg.h"

#include <cfloat>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>

#include "pkdg_kernels.cuh"

using namespace pkdg;

namespace {

constexpr int kMaxSlots = 8;

struct Slot {
    cudaStream_t st = nullptr;
    cudaEvent_t done = nullptr;
    bool busy = false;
    int32_t *pp_idx = nullptr, *pc_idx = nullptr;
    int64_t cap_pp = 0, cap_pc = 0;
    int32_t *first = nullptr, *count = nullptr;
    int64_t *pp_off = nullptr, *pc_off = nullptr;
    BucketDesc* desc = nullptr;
    int64_t cap_b = 0;
};

}  // namespace

struct pkdg_ctx {
    int device = 0;
    int num_sms = 0;
    float* cellq = nullptr;
    int64_t cellq_cap = 0;
    BucketDesc* desc = nullptr;
    int64_t desc_cap = 0;
    DevStats* stats = nullptr;
    unsigned int* counters = nullptr;  // [kMaxSlots + 1]
    Slot slots[kMaxSlots];
    int n_slots_live = 0;
    cudaEvent_t ev_ready = nullptr;
    cudaStream_t own_stream = nullptr;  // pkdg_gravity_eval_host
    float *e2e_xyzm = nullptr, *e2e_cells = nullptr, *e2e_out = nullptr;
    int64_t e2e_np = 0, e2e_nc = 0, e2e_no = 0;
    int64_t* scan_tmp = nullptr;
    int64_t scan_cap = 0;
    int2* gfc = nullptr;               // PKDG_PP_LEAVES: (first, count) of every bucket
    int64_t gfc_cap = 0;
    int32_t *g_first = nullptr, *g_count = nullptr;  // streamed variants: device copy of the bucket arrays
    int64_t g_first_cap = 0, g_count_cap = 0;
    cudaStream_t last_stream = nullptr;
    int64_t launches = 0;
    int64_t last_chunks = 1, last_buckets = 0;
    bool profiling = false;
    cudaEvent_t prof_ev[512] = {};
    int prof_n = 0;
    std::string err;
};

namespace {

pkdg_status fail(pkdg_ctx* ctx, pkdg_status s, const std::string& msg) {
    if (ctx) ctx->err = msg;
    return s;
}

#define CK(call)                                                                                   \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess)                                                                     \
            return fail(ctx, e_ == cudaErrorMemoryAllocation ? PKDG_ENOMEM : PKDG_ECUDA,           \
                        std::string(#call) + ": " + cudaGetErrorString(e_));                       \
    } while (0)

template <typename T>
pkdg_status ensure(pkdg_ctx* ctx, T** ptr, int64_t* cap, int64_t need) {
    if (need <= *cap) return PKDG_OK;
    if (*ptr) CK(cudaFree(*ptr));  // synchronises: documented ("grows on demand")
    *ptr = nullptr;
    *cap = 0;
    int64_t n = need + need / 8 + 64;
    CK(cudaMalloc((void**)ptr, sizeof(T) * (size_t)n));
    *cap = n;
    return PKDG_OK;
}

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

template <int WARPS, int MINB, bool NEWTON, int UNR>
pkdg_status launch_eval_t(pkdg_ctx* ctx, const EvalParams& p, cudaStream_t st) {
    int per_sm = 0;
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, pkdg_eval_kernel<WARPS, MINB, NEWTON, UNR>, WARPS * 32, 0));
    if (per_sm < 1) per_sm = 1;
    int64_t want = (p.n_buckets + WARPS - 1) / WARPS;
    int64_t grid = (int64_t)ctx->num_sms * per_sm;
    if (grid > want) grid = want;
    if (grid < 1) grid = 1;
    pkdg_eval_kernel<WARPS, MINB, NEWTON, UNR><<<(unsigned)grid, WARPS * 32, 0, st>>>(p);
    ctx->launches++;
    CK(cudaGetLastError());
    return PKDG_OK;
}

template <int WARPS, int MINB, bool NEWTON>
pkdg_status launch_eval3_t(pkdg_ctx* ctx, const EvalParams& p, cudaStream_t st) {
    auto kern = pkdg_eval3_kernel<WARPS, MINB, NEWTON>;
    const int smem = WARPS * (int)sizeof(WarpSmem3);
    static bool configured = false;  // per instantiation; the attribute is per function and sticky
    if (!configured) {
        CK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        CK(cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
        configured = true;
    }
    int per_sm = 0;
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, WARPS * 32, smem));
    if (per_sm < 1) per_sm = 1;
    int64_t want = (p.n_buckets + WARPS - 1) / WARPS;
    int64_t grid = (int64_t)ctx->num_sms * per_sm;
    if (grid > want) grid = want;
    if (grid < 1) grid = 1;
    kern<<<(unsigned)grid, WARPS * 32, smem, st>>>(p);
    ctx->launches++;
    CK(cudaGetLastError());
    return PKDG_OK;
}

// Tuning variants (flags bits 8..15).  0 = library default.
pkdg_status launch_eval(pkdg_ctx* ctx, const EvalParams& p, cudaStream_t st) {
    unsigned variant = (p.flags >> PKDG_VARIANT_SHIFT) & 0xffu;
    if ((p.flags & PKDG_PP_LEAVES) && variant == 1)
        return fail(ctx, PKDG_EINVAL, "PKDG_PP_LEAVES is not implemented by kernel variant 1 (generation 1)");
    switch (variant) {
        case 0: return launch_eval3_t<4, 3, false>(ctx, p, st);   // packed FP32x2, 168 registers, 12 warps / SM
        case 1: return launch_eval_t<4, 4, true, 2>(ctx, p, st);  // generation 1: scalar arithmetic (A/B reference)
        case 2: return launch_eval3_t<4, 4, false>(ctx, p, st);   // packed, 128 registers, 16 warps / SM
        case 3: return launch_eval3_t<4, 3, true>(ctx, p, st);    // packed, Newton step on the P-C rsqrt
        default: return fail(ctx, PKDG_EINVAL, "unknown kernel variant in flags bits 8..15");
    }
}

pkdg_status check_common(pkdg_ctx* ctx, const pkdg_particles* P, const pkdg_cells* C, const pkdg_buckets* B,
                         const pkdg_list* pp, const pkdg_list* pc, const float* out) {
    if (!ctx) return PKDG_EINVAL;
    if (!P || !B || !out) return fail(ctx, PKDG_EINVAL, "particles, buckets and out must not be NULL");
    if (P->n < 0 || B->n < 0 || P->n > 0x7fffffffLL) return fail(ctx, PKDG_EINVAL, "negative or too large size");
    if (P->n > 0 && !P->xyzm) return fail(ctx, PKDG_EINVAL, "particles->xyzm is NULL");
    if (B->n > 0 && (!B->first || !B->count)) return fail(ctx, PKDG_EINVAL, "buckets->first/count is NULL");
    if (!aligned16(P->xyzm) || !aligned16(out)) return fail(ctx, PKDG_EINVAL, "xyzm and out must be 16-byte aligned");
    bool has_pc = pc && pc->offsets;
    if (has_pc) {
        if (!C || C->n < 0 || C->n > 0x7fffffffLL) return fail(ctx, PKDG_EINVAL, "P-C list given without valid cells");
        if (C->n > 0 && !C->rec) return fail(ctx, PKDG_EINVAL, "cells->rec is NULL");
        if (C->stride_floats < PKDG_CELL_FLOATS) return fail(ctx, PKDG_EINVAL, "cells->stride_floats < 36");
    }
    return PKDG_OK;
}

void fill_params(EvalParams& p, pkdg_ctx* ctx, const float* xyzm, int64_t np, int64_t nc, float eps, uint32_t flags,
                 float* out) {
    p.xyzm = reinterpret_cast<const float4*>(xyzm);
    p.cellq = reinterpret_cast<const float4*>(ctx->cellq);
    p.out = reinterpret_cast<float4*>(out);
    p.stats = ctx->stats;
    p.n_particles = np;
    p.n_cells = nc;
    float h = 2.0f * eps;
    p.h2 = h * h;
    p.h2c = fmaxf(h * h, 1.0e-24f);
    p.hinv = h > 0.0f ? 1.0f / h : 0.0f;
    p.flags = flags;
}

pkdg_status prep_cells(pkdg_ctx* ctx, const pkdg_cells* C, float* dst, cudaStream_t st) {
    if (!C || C->n == 0) return PKDG_OK;
    const int threads = kPrepThreads;
    int64_t blocks = (C->n + threads - 1) / threads;
    pkdg_prep_cells_kernel<<<(unsigned)blocks, threads, 0, st>>>(C->rec, C->n, C->stride_floats, dst);
    ctx->launches++;
    CK(cudaGetLastError());
    return PKDG_OK;
}

// (first, count) records of all n buckets from DEVICE arrays (PKDG_PP_LEAVES)
pkdg_status build_gfc(pkdg_ctx* ctx, const int32_t* first, const int32_t* count, int64_t n, int64_t n_particles,
                      cudaStream_t st) {
    pkdg_status s = ensure(ctx, &ctx->gfc, &ctx->gfc_cap, n);
    if (s != PKDG_OK || n == 0) return s;
    pkdg_fc_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(first, count, n, n_particles, ctx->gfc);
    ctx->launches++;
    CK(cudaGetLastError());
    return PKDG_OK;
}

pkdg_status ensure_slots(pkdg_ctx* ctx, int n) {
    for (int i = ctx->n_slots_live; i < n; ++i) {
        CK(cudaStreamCreateWithFlags(&ctx->slots[i].st, cudaStreamNonBlocking));
        CK(cudaEventCreateWithFlags(&ctx->slots[i].done, cudaEventDisableTiming));
        ctx->n_slots_live = i + 1;
    }
    return PKDG_OK;
}

int64_t chunk_bounds_host(int64_t nb, const int64_t* pp_off, const int64_t* pc_off, int64_t max_entries,
                          int64_t* bounds) {
    int64_t nc = 0, b0 = 0;
    bounds[0] = 0;
    if (nb == 0) return 0;
    for (int64_t b = 0; b < nb; ++b) {
        int64_t pp = pp_off ? pp_off[b + 1] - pp_off[b0] : 0;
        int64_t pc = pc_off ? pc_off[b + 1] - pc_off[b0] : 0;
        if ((pp > max_entries || pc > max_entries) && b > b0) {
            bounds[++nc] = b;
            b0 = b;
        }
    }
    bounds[++nc] = nb;
    return nc;
}

}  // namespace

extern "C" {

pkdg_status pkdg_create(pkdg_ctx** out, int device) {
    if (!out) return PKDG_EINVAL;
    *out = nullptr;
    pkdg_ctx* ctx = new (std::nothrow) pkdg_ctx();
    if (!ctx) return PKDG_ENOMEM;
    ctx->device = device;
    cudaError_t e = cudaSetDevice(device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&ctx->num_sms, cudaDevAttrMultiProcessorCount, device);
    if (e == cudaSuccess) e = cudaMalloc((void**)&ctx->stats, sizeof(DevStats));
    if (e == cudaSuccess) e = cudaMalloc((void**)&ctx->counters, sizeof(unsigned int) * (kMaxSlots + 1));
    if (e == cudaSuccess) e = cudaMemset(ctx->stats, 0, sizeof(DevStats));
    if (e == cudaSuccess) e = cudaMemset(ctx->counters, 0, sizeof(unsigned int) * (kMaxSlots + 1));
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_ready, cudaEventDisableTiming);
    if (e != cudaSuccess) {
        fprintf(stderr, "pkdg_create: %s\n", cudaGetErrorString(e));
        delete ctx;
        return PKDG_ECUDA;
    }
    *out = ctx;
    return PKDG_OK;
}

pkdg_status pkdg_destroy(pkdg_ctx* ctx) {
    if (!ctx) return PKDG_OK;
    cudaSetDevice(ctx->device);
    cudaDeviceSynchronize();
    cudaFree(ctx->cellq); cudaFree(ctx->desc); cudaFree(ctx->stats); cudaFree(ctx->counters);
    cudaFree(ctx->e2e_xyzm); cudaFree(ctx->e2e_cells); cudaFree(ctx->e2e_out); cudaFree(ctx->scan_tmp);
    cudaFree(ctx->gfc); cudaFree(ctx->g_first); cudaFree(ctx->g_count);
    for (int i = 0; i < ctx->n_slots_live; ++i) {
        Slot& s = ctx->slots[i];
        cudaFree(s.pp_idx); cudaFree(s.pc_idx); cudaFree(s.first); cudaFree(s.count);
        cudaFree(s.pp_off); cudaFree(s.pc_off); cudaFree(s.desc);
        if (s.st) cudaStreamDestroy(s.st);
        if (s.done) cudaEventDestroy(s.done);
    }
    for (cudaEvent_t e : ctx->prof_ev)
        if (e) cudaEventDestroy(e);
    if (ctx->own_stream) cudaStreamDestroy(ctx->own_stream);
    if (ctx->ev_ready) cudaEventDestroy(ctx->ev_ready);
    delete ctx;
    return PKDG_OK;
}

pkdg_status pkdg_gravity_eval(pkdg_ctx* ctx, const pkdg_particles* P, const pkdg_cells* C, const pkdg_buckets* B,
                              const pkdg_list* pp, const pkdg_list* pc, float eps, uint32_t flags, float* out,
                              void* stream) {
    pkdg_status s = check_common(ctx, P, C, B, pp, pc, out);
    if (s != PKDG_OK) return s;
    cudaStream_t st = (cudaStream_t)stream;
    CK(cudaSetDevice(ctx->device));
    const bool has_pp = pp && pp->offsets, has_pc = pc && pc->offsets && C && C->n > 0;
    ctx->last_stream = st; ctx->last_chunks = 1; ctx->last_buckets = B->n;
    CK(cudaMemsetAsync(ctx->stats, 0, sizeof(DevStats), st));
    if (B->n == 0) return PKDG_OK;
    if ((s = ensure(ctx, &ctx->desc, &ctx->desc_cap, B->n)) != PKDG_OK) return s;
    if (has_pc) {
        if ((s = ensure(ctx, &ctx->cellq, &ctx->cellq_cap, C->n * kCellQFloats)) != PKDG_OK) return s;
        if ((s = prep_cells(ctx, C, ctx->cellq, st)) != PKDG_OK) return s;
    }
    {
        int threads = 256;
        int64_t blocks = (B->n + threads - 1) / threads;
        const bool leaves = has_pp && (flags & PKDG_PP_LEAVES);
        if (leaves && (s = build_gfc(ctx, B->first, B->count, B->n, P->n, st)) != PKDG_OK) return s;
        pkdg_pack_kernel<<<(unsigned)blocks, threads, 0, st>>>(B->first, B->count, has_pp ? pp->offsets : nullptr,
                                                             has_pc ? pc->offsets : nullptr, B->n, P->n, 0, 0,
                                                             ctx->desc, ctx->stats, ctx->counters + kMaxSlots,
                                                             leaves ? pp->idx : nullptr, ctx->gfc, B->n);
        ctx->launches++;
        CK(cudaGetLastError());
    }
    EvalParams p;
    fill_params(p, ctx, P->xyzm, P->n, has_pc ? C->n : 0, eps, flags, out);
    p.desc = ctx->desc;
    p.pp_idx = has_pp ? pp->idx : nullptr;
    p.pc_idx = has_pc ? pc->idx : nullptr;
    p.work_counter = ctx->counters + kMaxSlots;
    p.n_buckets = B->n;
    p.gfc = ctx->gfc;
    p.n_gbuckets = B->n;
    const bool prof = ctx->profiling && ctx->prof_n < 256;
    if (prof) {
        for (int i = 0; i < 2; ++i)
            if (!ctx->prof_ev[2 * ctx->prof_n + i]) CK(cudaEventCreate(&ctx->prof_ev[2 * ctx->prof_n + i]));
        CK(cudaEventRecord(ctx->prof_ev[2 * ctx->prof_n], st));
    }
    s = launch_eval(ctx, p, st);
    if (prof) {
        CK(cudaEventRecord(ctx->prof_ev[2 * ctx->prof_n + 1], st));
        ctx->prof_n++;
    }
    return s;
}

// out_host != NULL: the rows of every chunk (buckets are then known to be contiguous runs in ascending
// order, see pkdg_gravity_eval_host) are copied back on the chunk's stream right after its kernel, so
// the device->host traffic overlaps the host->device traffic of later chunks (PCIe is full duplex).
static pkdg_status streamed_impl(pkdg_ctx* ctx, const pkdg_particles* P, const pkdg_cells* C,
                                 const pkdg_buckets* Bh, const pkdg_list* pph, const pkdg_list* pch, float eps,
                                 uint32_t flags, float* out, int32_t n_streams, int64_t max_entries,
                                 void* stream, float* out_host) {
    pkdg_status s = check_common(ctx, P, C, Bh, pph, pch, out);
    if (s != PKDG_OK) return s;
    if (n_streams < 1 || n_streams > kMaxSlots) return fail(ctx, PKDG_EINVAL, "n_streams must be in 1..8");
    if (max_entries < 1) return fail(ctx, PKDG_EINVAL, "max_entries_per_chunk must be >= 1");
    cudaStream_t st = (cudaStream_t)stream;
    CK(cudaSetDevice(ctx->device));
    const bool has_pp = pph && pph->offsets, has_pc = pch && pch->offsets && C && C->n > 0;
    const int64_t nb = Bh->n;
    ctx->last_stream = st; ctx->last_buckets = nb; ctx->last_chunks = 0;
    CK(cudaMemsetAsync(ctx->stats, 0, sizeof(DevStats), st));
    if (nb == 0) return PKDG_OK;
    if ((s = ensure_slots(ctx, n_streams)) != PKDG_OK) return s;
    if (has_pc) {
        if ((s = ensure(ctx, &ctx->cellq, &ctx->cellq_cap, C->n * kCellQFloats)) != PKDG_OK) return s;
        if ((s = prep_cells(ctx, C, ctx->cellq, st)) != PKDG_OK) return s;
    }
    const bool leaves = has_pp && (flags & PKDG_PP_LEAVES);
    if (leaves) {  // leaf references may point at any bucket: all (first, count) pairs go to the device first
        if ((s = ensure(ctx, &ctx->g_first, &ctx->g_first_cap, nb)) != PKDG_OK) return s;
        if ((s = ensure(ctx, &ctx->g_count, &ctx->g_count_cap, nb)) != PKDG_OK) return s;
        CK(cudaMemcpyAsync(ctx->g_first, Bh->first, sizeof(int32_t) * nb, cudaMemcpyHostToDevice, st));
        CK(cudaMemcpyAsync(ctx->g_count, Bh->count, sizeof(int32_t) * nb, cudaMemcpyHostToDevice, st));
        if ((s = build_gfc(ctx, ctx->g_first, ctx->g_count, nb, P->n, st)) != PKDG_OK) return s;
    }
    CK(cudaEventRecord(ctx->ev_ready, st));
    int64_t* bounds = (int64_t*)malloc(sizeof(int64_t) * (size_t)(nb + 1));
    if (!bounds) return fail(ctx, PKDG_ENOMEM, "host malloc of chunk bounds failed");
    const int64_t nchunk = chunk_bounds_host(nb, has_pp ? pph->offsets : nullptr, has_pc ? pch->offsets : nullptr,
                                             max_entries, bounds);
    ctx->last_chunks = nchunk;
    pkdg_status rc = PKDG_OK;
    for (int i = 0; i < n_streams; ++i) {
        if (cudaStreamWaitEvent(ctx->slots[i].st, ctx->ev_ready, 0) != cudaSuccess) rc = PKDG_ECUDA;
        ctx->slots[i].busy = false;
    }
    for (int64_t ic = 0; ic < nchunk && rc == PKDG_OK; ++ic) {
        Slot& sl = ctx->slots[ic % n_streams];
        const int64_t b0 = bounds[ic], b1 = bounds[ic + 1], cb = b1 - b0;
        const int64_t pbase = has_pp ? pph->offsets[b0] : 0, plen = has_pp ? pph->offsets[b1] - pbase : 0;
        const int64_t cbase = has_pc ? pch->offsets[b0] : 0, clen = has_pc ? pch->offsets[b1] - cbase : 0;
        // bounded in-flight work: a slot is reused only after its previous chunk is done
        if (sl.busy && cudaEventSynchronize(sl.done) != cudaSuccess) { rc = PKDG_ECUDA; break; }
        if ((rc = ensure(ctx, &sl.pp_idx, &sl.cap_pp, plen)) != PKDG_OK) break;
        if ((rc = ensure(ctx, &sl.pc_idx, &sl.cap_pc, clen)) != PKDG_OK) break;
        if (cb + 1 > sl.cap_b) {
            int64_t c1 = 0, c2 = 0, c3 = 0, c4 = 0, c5 = 0;
            cudaFree(sl.first); cudaFree(sl.count); cudaFree(sl.pp_off); cudaFree(sl.pc_off); cudaFree(sl.desc);
            sl.first = sl.count = nullptr; sl.pp_off = sl.pc_off = nullptr; sl.desc = nullptr; sl.cap_b = 0;
            if ((rc = ensure(ctx, &sl.first, &c1, cb + 1)) != PKDG_OK) break;
            if ((rc = ensure(ctx, &sl.count, &c2, cb + 1)) != PKDG_OK) break;
            if ((rc = ensure(ctx, &sl.pp_off, &c3, cb + 1)) != PKDG_OK) break;
            if ((rc = ensure(ctx, &sl.pc_off, &c4, cb + 1)) != PKDG_OK) break;
            if ((rc = ensure(ctx, &sl.desc, &c5, cb + 1)) != PKDG_OK) break;
            sl.cap_b = c1;
        }
        cudaError_t e = cudaMemcpyAsync(sl.first, Bh->first + b0, sizeof(int32_t) * cb, cudaMemcpyHostToDevice, sl.st);
        if (e == cudaSuccess) e = cudaMemcpyAsync(sl.count, Bh->count + b0, sizeof(int32_t) * cb, cudaMemcpyHostToDevice, sl.st);
        if (e == cudaSuccess && has_pp) {
            e = cudaMemcpyAsync(sl.pp_off, pph->offsets + b0, sizeof(int64_t) * (cb + 1), cudaMemcpyHostToDevice, sl.st);
            if (e == cudaSuccess && plen)
                e = cudaMemcpyAsync(sl.pp_idx, pph->idx + pbase, sizeof(int32_t) * plen, cudaMemcpyHostToDevice, sl.st);
        }
        if (e == cudaSuccess && has_pc) {
            e = cudaMemcpyAsync(sl.pc_off, pch->offsets + b0, sizeof(int64_t) * (cb + 1), cudaMemcpyHostToDevice, sl.st);
            if (e == cudaSuccess && clen)
                e = cudaMemcpyAsync(sl.pc_idx, pch->idx + cbase, sizeof(int32_t) * clen, cudaMemcpyHostToDevice, sl.st);
        }
        if (e != cudaSuccess) { rc = fail(ctx, PKDG_ECUDA, std::string("chunk copy: ") + cudaGetErrorString(e)); break; }
        unsigned int* counter = ctx->counters + (ic % n_streams);
        int threads = 256;
        pkdg_pack_kernel<<<(unsigned)((cb + threads - 1) / threads), threads, 0, sl.st>>>(
            sl.first, sl.count, has_pp ? sl.pp_off : nullptr, has_pc ? sl.pc_off : nullptr, cb, P->n, pbase, cbase,
            sl.desc, ctx->stats, counter, leaves ? sl.pp_idx : nullptr, ctx->gfc, nb);
        ctx->launches++;
        EvalParams p;
        fill_params(p, ctx, P->xyzm, P->n, has_pc ? C->n : 0, eps, flags, out);
        p.desc = sl.desc;
        p.pp_idx = sl.pp_idx;
        p.pc_idx = sl.pc_idx;
        p.work_counter = counter;
        p.n_buckets = cb;
        p.gfc = ctx->gfc;
        p.n_gbuckets = nb;
        if ((rc = launch_eval(ctx, p, sl.st)) != PKDG_OK) break;
        if (out_host) {
            const int64_t r0 = Bh->first[b0], r1 = (int64_t)Bh->first[b1 - 1] + Bh->count[b1 - 1];
            if (r1 > r0 && cudaMemcpyAsync(out_host + 4 * r0, out + 4 * r0, sizeof(float) * 4 * (size_t)(r1 - r0),
                                           cudaMemcpyDeviceToHost, sl.st) != cudaSuccess) { rc = PKDG_ECUDA; break; }
        }
        if (cudaEventRecord(sl.done, sl.st) != cudaSuccess) { rc = PKDG_ECUDA; break; }
        sl.busy = true;
    }
    free(bounds);
    for (int i = 0; i < n_streams; ++i)
        if (ctx->slots[i].busy && cudaStreamWaitEvent(st, ctx->slots[i].done, 0) != cudaSuccess && rc == PKDG_OK)
            rc = PKDG_ECUDA;
    if (rc == PKDG_ECUDA && ctx->err.empty()) ctx->err = cudaGetErrorString(cudaGetLastError());
    return rc;
}

pkdg_status pkdg_gravity_eval_streamed(pkdg_ctx* ctx, const pkdg_particles* P, const pkdg_cells* C,
                                       const pkdg_buckets* Bh, const pkdg_list* pph, const pkdg_list* pch, float eps,
                                       uint32_t flags, float* out, int32_t n_streams, int64_t max_entries,
                                       void* stream) {
    return streamed_impl(ctx, P, C, Bh, pph, pch, eps, flags, out, n_streams, max_entries, stream, nullptr);
}

pkdg_status pkdg_gravity_eval_host(pkdg_ctx* ctx, const pkdg_particles* Ph, const pkdg_cells* Ch,
                                   const pkdg_buckets* Bh, const pkdg_list* pph, const pkdg_list* pch, float eps,
                                   uint32_t flags, float* out_host, int32_t n_streams, int64_t max_entries) {
    pkdg_status s = check_common(ctx, Ph, Ch, Bh, pph, pch, out_host);
    if (s != PKDG_OK) return s;
    CK(cudaSetDevice(ctx->device));
    if (!ctx->own_stream) CK(cudaStreamCreateWithFlags(&ctx->own_stream, cudaStreamNonBlocking));
    cudaStream_t st = ctx->own_stream;
    const bool has_pc = pch && pch->offsets && Ch && Ch->n > 0;
    if ((s = ensure(ctx, &ctx->e2e_xyzm, &ctx->e2e_np, Ph->n * 4)) != PKDG_OK) return s;
    if ((s = ensure(ctx, &ctx->e2e_out, &ctx->e2e_no, Ph->n * 4)) != PKDG_OK) return s;
    if (Ph->n) CK(cudaMemcpyAsync(ctx->e2e_xyzm, Ph->xyzm, sizeof(float) * 4 * Ph->n, cudaMemcpyHostToDevice, st));
    pkdg_cells Cd = {nullptr, 0, PKDG_CELL_FLOATS};
    if (has_pc) {
        if ((s = ensure(ctx, &ctx->e2e_cells, &ctx->e2e_nc, Ch->n * (int64_t)Ch->stride_floats)) != PKDG_OK) return s;
        CK(cudaMemcpyAsync(ctx->e2e_cells, Ch->rec, sizeof(float) * Ch->n * Ch->stride_floats, cudaMemcpyHostToDevice, st));
        Cd.rec = ctx->e2e_cells; Cd.n = Ch->n; Cd.stride_floats = Ch->stride_floats;
    }
    if (flags & PKDG_ACCUMULATE) {
        if (Ph->n) CK(cudaMemcpyAsync(ctx->e2e_out, out_host, sizeof(float) * 4 * Ph->n, cudaMemcpyHostToDevice, st));
    } else if (Ph->n) {
        CK(cudaMemsetAsync(ctx->e2e_out, 0, sizeof(float) * 4 * Ph->n, st));  // rows in no bucket come back as 0
    }
    pkdg_particles Pd = {ctx->e2e_xyzm, Ph->n};
    // tree-ordered input (every bucket starts where the previous one ends, together they cover all rows):
    // each chunk's rows go back as soon as they are done; anything else: one copy at the end
    bool tiled = Bh->n > 0 && Bh->first[0] == 0;
    for (int64_t b = 0; tiled && b < Bh->n; ++b) {
        const int64_t end = (int64_t)Bh->first[b] + Bh->count[b];
        tiled = Bh->count[b] >= 0 && end == (b + 1 < Bh->n ? (int64_t)Bh->first[b + 1] : Ph->n);
    }
    s = streamed_impl(ctx, &Pd, has_pc ? &Cd : nullptr, Bh, pph, has_pc ? pch : nullptr, eps, flags, ctx->e2e_out,
                      n_streams, max_entries, st, tiled ? out_host : nullptr);
    if (s != PKDG_OK) return s;
    if (!tiled && Ph->n)
        CK(cudaMemcpyAsync(out_host, ctx->e2e_out, sizeof(float) * 4 * Ph->n, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    return PKDG_OK;
}

pkdg_status pkdg_pack_export(pkdg_ctx* ctx, int64_t n_buckets, const pkdg_list* list, int64_t* tile_offsets,
                             int32_t* tiles, int64_t tile_capacity, void* stream) {
    if (!ctx) return PKDG_EINVAL;
    if (!list || !list->offsets || n_buckets < 0) return fail(ctx, PKDG_EINVAL, "list/offsets NULL or n_buckets < 0");
    cudaStream_t st = (cudaStream_t)stream;
    CK(cudaSetDevice(ctx->device));
    pkdg_status s;
    int64_t* toff = tile_offsets;
    if (!toff) {
        if ((s = ensure(ctx, &ctx->scan_tmp, &ctx->scan_cap, n_buckets + 1)) != PKDG_OK) return s;
        toff = ctx->scan_tmp;
    }
    if (n_buckets > 0) {
        int threads = 256;
        pkdg_tile_count_kernel<<<(unsigned)((n_buckets + threads - 1) / threads), threads, 0, st>>>(list->offsets,
                                                                                                  n_buckets, toff);
        ctx->launches++;
    }
    pkdg_scan_kernel<<<1, 1024, 0, st>>>(toff, n_buckets);
    ctx->launches++;
    if (tiles && n_buckets > 0 && tile_capacity > 0) {
        if (!list->idx) return fail(ctx, PKDG_EINVAL, "list->idx is NULL");
        pkdg_tiles_kernel<<<ctx->num_sms * 8, 256, 0, st>>>(list->offsets, list->idx, n_buckets, toff, tiles,
                                                            tile_capacity);
        ctx->launches++;
    }
    CK(cudaGetLastError());
    return PKDG_OK;
}

pkdg_status pkdg_chunk_bounds(int64_t n_buckets, const int64_t* pp_off, const int64_t* pc_off, int64_t max_entries,
                              int64_t* bounds, int64_t* n_chunks) {
    if (n_buckets < 0 || !bounds || !n_chunks || max_entries < 1) return PKDG_EINVAL;
    *n_chunks = chunk_bounds_host(n_buckets, pp_off, pc_off, max_entries, bounds);
    return PKDG_OK;
}

pkdg_status pkdg_prepare_cells_export(pkdg_ctx* ctx, const pkdg_cells* C, float* out, void* stream) {
    if (!ctx) return PKDG_EINVAL;
    if (!C || !out || C->n < 0 || (C->n > 0 && !C->rec) || C->stride_floats < PKDG_CELL_FLOATS)
        return fail(ctx, PKDG_EINVAL, "bad cells or out");
    CK(cudaSetDevice(ctx->device));
    return prep_cells(ctx, C, out, (cudaStream_t)stream);
}

pkdg_status pkdg_get_stats(pkdg_ctx* ctx, pkdg_stats* out) {
    if (!ctx || !out) return PKDG_EINVAL;
    CK(cudaSetDevice(ctx->device));
    CK(cudaStreamSynchronize(ctx->last_stream));
    DevStats h;
    CK(cudaMemcpy(&h, ctx->stats, sizeof(DevStats), cudaMemcpyDeviceToHost));
    out->n_buckets = ctx->last_buckets;
    out->interactions_pp = (int64_t)h.interactions_pp;
    out->interactions_pc = (int64_t)h.interactions_pc;
    out->tiles_pp = (int64_t)h.tiles_pp;
    out->tiles_pc = (int64_t)h.tiles_pc;
    out->bad_entries = (int64_t)h.bad_entries;
    out->chunks = ctx->last_chunks;
    return h.bad_entries ? fail(ctx, PKDG_EBADLIST, "validation found malformed buckets or list entries") : PKDG_OK;
}

pkdg_status pkdg_profile_enable(pkdg_ctx* ctx, int32_t on) {
    if (!ctx) return PKDG_EINVAL;
    ctx->profiling = on != 0;
    return PKDG_OK;
}

pkdg_status pkdg_profile_read(pkdg_ctx* ctx, int64_t* n, double* ms_total) {
    if (!ctx || !n || !ms_total) return PKDG_EINVAL;
    CK(cudaSetDevice(ctx->device));
    double tot = 0;
    for (int i = 0; i < ctx->prof_n; ++i) {
        float ms = 0;
        CK(cudaEventSynchronize(ctx->prof_ev[2 * i + 1]));
        CK(cudaEventElapsedTime(&ms, ctx->prof_ev[2 * i], ctx->prof_ev[2 * i + 1]));
        tot += ms;
    }
    *n = ctx->prof_n;
    *ms_total = tot;
    ctx->prof_n = 0;
    return PKDG_OK;
}

int64_t pkdg_launch_count(const pkdg_ctx* ctx) { return ctx ? ctx->launches : 0; }

const char* pkdg_status_string(pkdg_status s) {
    switch (s) {
        case PKDG_OK: return "PKDG_OK";
        case PKDG_EINVAL: return "PKDG_EINVAL: invalid argument";
        case PKDG_ECUDA: return "PKDG_ECUDA: CUDA runtime error";
        case PKDG_ENOMEM: return "PKDG_ENOMEM: out of memory";
        case PKDG_EBADLIST: return "PKDG_EBADLIST: malformed buckets or lists";
        default: return "unknown pkdg_status";
    }
}

const char* pkdg_last_error(const pkdg_ctx* ctx) { return ctx ? ctx->err.c_str() : "no context"; }

void pkdg_version(int32_t* major, int32_t* minor) {
    if (major) *major = PKDG_VERSION_MAJOR;
    if (minor) *minor = PKDG_VERSION_MINOR;
}

pkdg_status pkdg_fma_probe(pkdg_ctx* ctx, int32_t mode, int64_t iters, float* ms_host, double* flops_host) {
    if (!ctx || !ms_host || !flops_host || iters < 1) return PKDG_EINVAL;
    if (mode < 0 || mode > 5) return fail(ctx, PKDG_EINVAL, "probe mode must be in 0..5");
    CK(cudaSetDevice(ctx->device));
    const int threads = mode == 0 ? 256 : 128, blocks = ctx->num_sms * (mode == 0 ? 8 : 4);
    float *buf = nullptr, *in = nullptr;
    CK(cudaMalloc((void**)&buf, sizeof(float4) * threads * blocks));
    // input: 1024 operands around 0.5; 32 synthetic cell records (COM, M, s, small moments); 2 sinks
    float h[2048];
    for (int i = 0; i < 1024; ++i) h[i] = 0.5f + 0.001f * (float)(i % 97);
    float* hc = h + 1024;
    for (int i = 0; i < 32 * 32; ++i) hc[i] = 0.01f * (float)(i % 13) - 0.03f;
    for (int l = 0; l < 32; ++l) {
        hc[l * 32 + 0] = 0.1f * l; hc[l * 32 + 1] = 0.2f; hc[l * 32 + 2] = 0.3f; hc[l * 32 + 3] = 1.0f;
        hc[l * 32 + 4] = 0.05f;
    }
    const float tgt[8] = {5.f, 6.f, 7.f, 0.f, -5.f, 6.f, -7.f, 0.f};
    CK(cudaMalloc((void**)&in, sizeof(h) + sizeof(tgt)));
    CK(cudaMemcpy(in, h, sizeof(h), cudaMemcpyHostToDevice));
    CK(cudaMemcpy(in + 2048, tgt, sizeof(tgt), cudaMemcpyHostToDevice));
    const float4* cells = reinterpret_cast<const float4*>(in + 1024);
    const float4* tg = reinterpret_cast<const float4*>(in + 2048);
    auto launch = [&](int64_t n) {
        switch (mode) {
            case 0: pkdg_fma_probe_kernel<<<blocks, threads>>>(buf, n, 0.999f, 0.001f); break;
            case 1: pkdg_rf_probe_kernel<1><<<blocks, threads>>>(in, buf, n); break;
            case 2: pkdg_rf_probe_kernel<2><<<blocks, threads>>>(in, buf, n); break;
            case 3: pkdg_rf_probe_kernel<3><<<blocks, threads>>>(in, buf, n); break;
            case 4: pkdg_pc_probe_kernel<false><<<blocks, threads>>>(cells, tg, reinterpret_cast<float4*>(buf), n); break;
            default: pkdg_pc_probe_kernel<true><<<blocks, threads>>>(cells, tg, reinterpret_cast<float4*>(buf), n); break;
        }
    };
    if (mode >= 4) iters = (iters + 1) & ~(int64_t)1;
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0));
    CK(cudaEventCreate(&e1));
    launch(16);  // warm-up
    CK(cudaEventRecord(e0, 0));
    launch(iters);
    CK(cudaEventRecord(e1, 0));
    CK(cudaEventSynchronize(e1));
    ctx->launches += 2;
    CK(cudaGetLastError());
    CK(cudaEventElapsedTime(ms_host, e0, e1));
    const double lanes = (double)threads * blocks;
    switch (mode) {
        case 0: case 1: *flops_host = 2.0 * 64.0 * (double)iters * lanes; break;  // 64 FFMA per trip
        case 2: case 3: *flops_host = 4.0 * 64.0 * (double)iters * lanes; break;  // 64 FFMA2 per trip
        case 4: *flops_host = 2.0 * 196.0 * (double)iters * lanes; break;         // 2 sinks per trip
        default: *flops_host = 2.0 * 187.0 * (double)iters * lanes; break;        // 1 sink pair per trip
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    CK(cudaFree(buf));
    CK(cudaFree(in));
    return PKDG_OK;
}

pkdg_status pkdg_fma_peak_probe(pkdg_ctx* ctx, int64_t iters, float* ms_host, double* flops_host) {
    return pkdg_fma_probe(ctx, PKDG_PROBE_FFMA_CONST, iters, ms_host, flops_host);
}

}  // extern "C"
