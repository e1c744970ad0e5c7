// pkdg.cu -- host side of the C ABI declared in include/pkdg.h.  No CPU fallback exists: every
// entry point either runs the CUDA kernels of pkdg_kernels.cuh or returns an error.
#include "../../include/pkdg.h"

#include <cfloat>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <string>

#include "pkdg_kernels.cuh"
#include "pkdg_fmm.cuh"

using namespace pkdg;

namespace {

constexpr int kMaxSlots = 8;
// Conditioning threshold: a sink goes to the fp64 fix-up kernel
// when sqrt(sum_j |a_ij|^2) > kappa2 |a_i|.  Measured fp32 error <= 1.2e-6 sqrt(S2) / |a| over 1.3e7 sinks, so
// kappa2 = 6 keeps the fp32 path below 7e-6 of |a_i|, a third of the 2e-5 tolerance.
constexpr float kDefaultKappa2 = 6.0f;

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
    int4* fixq = nullptr;       // fix-up queue of the chunk in flight on this slot
    int64_t fixq_cap = 0;
    int32_t *gfirst = nullptr, *gn = nullptr;   // group-shared lists: the chunk's groups
    int64_t cap_g = 0, cap_off = 0;
};

}  // namespace

static thread_local std::string g_create_err;   // why the last pkdg_create / pkdg_gravity_eval_static of this thread failed

// ------------------------------------------------------------------------------------------------
// Workspace of pkdg_gravity_eval_static: the one entry point for callers that must not allocate device memory
// (include/pkdg.h says who they are).  A fixed array in the library's device image instead of cudaMalloc'ed
// buffers; every GPU that loads this module carries it until the process ends.  On the HOST the name
// g_static_scratch is only a handle for the runtime: its device address comes from cudaGetSymbolAddress, once
// per device (static_setup), and only that address is ever handed to a kernel.
//   [0, 256)    DevStats (the packer adds to it; nobody reads it back here)
//   [256, 512)  work counter of the evaluation kernel, length of the fix-up queue
//   then        bucket descriptors | normalised cell records | fix-up queue
// ------------------------------------------------------------------------------------------------
namespace {
constexpr size_t kStOffStats = 0, kStOffCounters = 256, kStOffDesc = 512;
constexpr size_t kStOffCellq = kStOffDesc + sizeof(BucketDesc) * PKDG_STATIC_MAX_BUCKETS;
constexpr size_t kStOffFixq = kStOffCellq + sizeof(float) * kCellQFloats * PKDG_STATIC_MAX_CELLS;
constexpr int64_t kStFixCap = PKDG_STATIC_MAX_BUCKETS + PKDG_STATIC_MAX_PARTICLES / kTMax + 16;
constexpr size_t kStBytes = kStOffFixq + sizeof(int4) * kStFixCap;
static_assert(kStBytes == PKDG_STATIC_SCRATCH_BYTES, "include/pkdg.h states the size of the static workspace");
static_assert(sizeof(DevStats) <= 256 && kStOffCellq % 256 == 0 && kStOffFixq % 256 == 0, "sections stay 256-byte aligned");
}  // namespace
static __device__ __align__(256) unsigned char g_static_scratch[kStBytes];

struct pkdg_ctx {
    int device = 0;
    int num_sms = 0;
    float* cellq = nullptr;
    int64_t cellq_cap = 0;
    BucketDesc* desc = nullptr;
    int64_t desc_cap = 0;
    DevStats* stats = nullptr;
    unsigned int* counters = nullptr;  // [2 (kMaxSlots + 1) + 1]: work counters, fix-up queue lengths, C-C / C-P kernel
    int4* fixq = nullptr;              // fix-up queue of the resident call
    int64_t fixq_cap = 0;
    float kappa2 = kDefaultKappa2;     // PKDG_OPT_KAPPA2
    unsigned long long fix_entries = 0, fix_calls = 0;
    Slot slots[kMaxSlots];
    int n_slots_live = 0;
    cudaEvent_t ev_ready = nullptr;
    cudaStream_t own_stream = nullptr;  // pkdg_gravity_eval_host
    float *e2e_xyzm = nullptr, *e2e_cells = nullptr, *e2e_out = nullptr;
    int64_t e2e_np = 0, e2e_nc = 0, e2e_no = 0;
    int64_t* scan_tmp = nullptr;
    int64_t scan_cap = 0;
    // pkdg_gravity_eval_tree_host: device copies of the tree and the lists built from it
    int32_t *t_first = nullptr, *t_count = nullptr, *t_end = nullptr, *t_isleaf = nullptr, *t_rank = nullptr, *t_sink = nullptr;
    float *t_bblo = nullptr, *t_bbhi = nullptr;
    int64_t t_cap[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    int32_t *t_bfirst = nullptr, *t_bcount = nullptr, *t_ppi = nullptr, *t_pci = nullptr;
    int64_t *t_ppo = nullptr, *t_pco = nullptr;
    int64_t t_bcap[6] = {0, 0, 0, 0, 0, 0};
    cudaEvent_t t_ev[2] = {nullptr, nullptr};
    WalkNode* wnodes = nullptr;        // pkdg_build_lists_*: one 64-byte record per tree cell
    int64_t wnodes_cap = 0;
    int2* gfc = nullptr;               // PKDG_PP_LEAVES: (first, count) of every bucket
    int64_t gfc_cap = 0;
    int32_t *g_first = nullptr, *g_count = nullptr;  // streamed variants: device copy of the bucket arrays
    int64_t g_first_cap = 0, g_count_cap = 0;
    cudaStream_t last_stream = nullptr;
    // CTAs per SM of the two instantiations (particle lists / PKDG_PP_LEAVES) of the bucket and of the group kernel;
    // 0 = the dynamic shared-memory opt-in has not been made on this context's device yet
    int evalb_per_sm[2] = {0, 0};
    int evalg_per_sm[2] = {0, 0};
    int64_t launches = 0;
    int64_t last_chunks = 1, last_buckets = 0;
    bool profiling = false;
    cudaEvent_t prof_ev[3 * 256] = {};  // per recorded call: before / after the evaluation kernel, after the fix-up
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

// The evaluation kernels need more than the default 48 KB of dynamic shared memory.  Function attributes are per
// device, so the opt-in is made once per context (a pkdg_ctx is bound to one device).
constexpr int kBucketWarps = 4;      // bucket kernel: one bucket per warp
#ifndef PKDG_B_MINB
#define PKDG_B_MINB 5
#endif
constexpr int kBucketMinBlocks = PKDG_B_MINB;  // 96 registers per thread: 20 warps per SM

template <bool LEAF>
pkdg_status launch_evalb_t(pkdg_ctx* ctx, const EvalParams& p, cudaStream_t st) {
    auto kern = pkdg_evalb_kernel<kBucketWarps, kBucketMinBlocks, LEAF>;
    const int smem = kBucketWarps * (int)sizeof(WarpSmemB);
    int& per_sm = ctx->evalb_per_sm[LEAF ? 1 : 0];
    if (per_sm == 0) {
        CK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        CK(cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
        CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, kBucketWarps * 32, smem));
        if (per_sm < 1) per_sm = 1;
    }
    int64_t want = (p.n_buckets + kBucketWarps - 1) / kBucketWarps;
    int64_t grid = (int64_t)ctx->num_sms * per_sm;
    if (grid > want) grid = want;
    if (grid < 1) grid = 1;
    kern<<<(unsigned)grid, kBucketWarps * 32, smem, st>>>(p);
    ctx->launches++;
    CK(cudaGetLastError());
    return PKDG_OK;
}

pkdg_status launch_eval(pkdg_ctx* ctx, const EvalParams& p, cudaStream_t st) {
    return (p.flags & PKDG_PP_LEAVES) ? launch_evalb_t<true>(ctx, p, st) : launch_evalb_t<false>(ctx, p, st);
}

constexpr int kGroupWarps = 4;      // warps per CTA of the group kernel (one group per warp)
constexpr int kGroupMinBlocks = 5;  // 92 registers per thread: 20 warps per SM (four CTAs at 115 registers: 1.2 % slower)

template <bool LEAF>
pkdg_status launch_eval_groups_t(pkdg_ctx* ctx, const EvalParams& p, cudaStream_t st) {
    auto kern = pkdg_evalg_kernel<kGroupWarps, kGroupMinBlocks, LEAF>;
    const int smem = kGroupWarps * (int)sizeof(WarpSmemG);
    int& per_sm = ctx->evalg_per_sm[LEAF ? 1 : 0];
    if (per_sm == 0) {
        CK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        CK(cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
        CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, kGroupWarps * 32, smem));
        if (per_sm < 1) per_sm = 1;
    }
    int64_t want = (p.n_groups + kGroupWarps - 1) / kGroupWarps;
    int64_t grid = (int64_t)ctx->num_sms * per_sm;
    if (grid > want) grid = want;
    if (grid < 1) grid = 1;
    kern<<<(unsigned)grid, kGroupWarps * 32, smem, st>>>(p);
    ctx->launches++;
    CK(cudaGetLastError());
    return PKDG_OK;
}

// Group-shared lists: one warp per group, one lane per sink pair (pkdg_evalg_kernel).
pkdg_status launch_eval_groups(pkdg_ctx* ctx, const EvalParams& p, cudaStream_t st) {
    return (p.flags & PKDG_PP_LEAVES) ? launch_eval_groups_t<true>(ctx, p, st) : launch_eval_groups_t<false>(ctx, p, st);
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
    p.eps = eps;
    p.h2c = fmaxf(h * h, 1.0e-24f);
    p.flags = flags;
    p.cells_raw = nullptr;
    p.cells_stride = PKDG_CELL_FLOATS;
    p.fix_k = (flags & PKDG_NO_FIXUP) ? -1.0f : (flags & PKDG_FIXUP_ALL) ? 0.0f : ctx->kappa2 * ctx->kappa2;
    p.fix_queue = nullptr;
    p.fix_count = nullptr;
    p.fix_cap = 0;
    p.g_first = nullptr;
    p.g_n = nullptr;
    p.n_groups = 0;
    p.g_base = 0;
}

// Queue capacity that cannot overflow: one entry per (bucket, pass of 16 sinks) at most.
// PKDG_VALIDATE: value-range and geometry contract of include/pkdg.h, counted into the statistics.
pkdg_status launch_validate(pkdg_ctx* ctx, const EvalParams& p, bool values, cudaStream_t st) {
    if (values) {
        pkdg_validate_values_kernel<<<ctx->num_sms * 8, 256, 0, st>>>(p.xyzm, p.n_particles, p.cells_raw,
                                                                     p.cells_raw ? p.n_cells : 0, p.cells_stride, p.stats);
        ctx->launches++;
    }
    if (p.n_cells > 0 && p.pc_idx) {
        pkdg_validate_pairs_kernel<<<ctx->num_sms * 8, 256, 0, st>>>(p);
        ctx->launches++;
    }
    CK(cudaGetLastError());
    return PKDG_OK;
}

int64_t fix_capacity(int64_t n_buckets, int64_t n_particles) { return n_buckets + n_particles / kTMax + 16; }

// The fp64 fix-up kernel over the queue the evaluation kernel just filled (same stream).  Its grid is fixed
// (the queue length is known only on the device); with an empty queue every warp leaves at once.
pkdg_status launch_fixup(pkdg_ctx* ctx, const EvalParams& p, cudaStream_t st) {
    if (p.fix_k < 0.0f) return PKDG_OK;
    int64_t grid = p.n_buckets < 1 ? 1 : p.n_buckets;   // one CTA per queue entry, persistent beyond 16 per SM
    const int64_t full = (int64_t)ctx->num_sms * 16;
    if (grid > full) grid = full;
    pkdg_fixup_kernel<<<(unsigned)grid, kFixThreads, 0, st>>>(p);
    ctx->launches++;
    CK(cudaGetLastError());
    return PKDG_OK;
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
    if (e == cudaSuccess) e = cudaMalloc((void**)&ctx->counters, sizeof(unsigned int) * (2 * (kMaxSlots + 1) + 1));
    if (e == cudaSuccess) e = cudaMemset(ctx->stats, 0, sizeof(DevStats));
    if (e == cudaSuccess) e = cudaMemset(ctx->counters, 0, sizeof(unsigned int) * (2 * (kMaxSlots + 1) + 1));
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_ready, cudaEventDisableTiming);
    if (e != cudaSuccess) {
        g_create_err = std::string("pkdg_create: ") + cudaGetErrorString(e);   // read with pkdg_last_error(NULL)
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
    cudaFree(ctx->t_first); cudaFree(ctx->t_count); cudaFree(ctx->t_end); cudaFree(ctx->t_isleaf); cudaFree(ctx->t_rank);
    cudaFree(ctx->t_sink); cudaFree(ctx->t_bblo); cudaFree(ctx->t_bbhi); cudaFree(ctx->t_bfirst); cudaFree(ctx->t_bcount);
    cudaFree(ctx->t_ppi); cudaFree(ctx->t_pci); cudaFree(ctx->t_ppo); cudaFree(ctx->t_pco);
    for (cudaEvent_t e : ctx->t_ev)
        if (e) cudaEventDestroy(e);
    cudaFree(ctx->gfc); cudaFree(ctx->wnodes); cudaFree(ctx->g_first); cudaFree(ctx->g_count); cudaFree(ctx->fixq);
    for (int i = 0; i < ctx->n_slots_live; ++i) {
        Slot& s = ctx->slots[i];
        cudaFree(s.pp_idx); cudaFree(s.pc_idx); cudaFree(s.first); cudaFree(s.count);
        cudaFree(s.pp_off); cudaFree(s.pc_off); cudaFree(s.desc); cudaFree(s.fixq); cudaFree(s.gfirst); cudaFree(s.gn);
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

// Sinks are buckets [b0, b1) of Bfull; the lists have b1 - b0 + 1 offsets; P-P leaf references index Bfull.
// G != NULL (group-shared lists): the lists have G->n + 1 offsets and the range must be all buckets.
static pkdg_status resident_impl(pkdg_ctx* ctx, const pkdg_particles* P, const pkdg_cells* C, const pkdg_buckets* Bfull,
                                 int64_t b0, int64_t b1, const pkdg_groups* G, const pkdg_list* pp, const pkdg_list* pc,
                                 float eps, uint32_t flags, float* out, void* stream, bool reset_stats = true) {
    pkdg_status s = check_common(ctx, P, C, Bfull, pp, pc, out);
    if (s != PKDG_OK) return s;
    if (G && (G->n < 0 || (G->n > 0 && (!G->first_bucket || !G->n_buckets))))
        return fail(ctx, PKDG_EINVAL, "groups->first_bucket / n_buckets is NULL or n < 0");
    if (b0 < 0 || b1 < b0 || b1 > Bfull->n) return fail(ctx, PKDG_EINVAL, "bucket range outside [0, buckets->n]");
    const pkdg_buckets Bsub = {Bfull->first ? Bfull->first + b0 : nullptr, Bfull->count ? Bfull->count + b0 : nullptr, b1 - b0};
    const pkdg_buckets* B = &Bsub;
    cudaStream_t st = (cudaStream_t)stream;
    CK(cudaSetDevice(ctx->device));
    const bool has_pp = pp && pp->offsets, has_pc = pc && pc->offsets && C && C->n > 0;
    ctx->last_stream = st; ctx->last_chunks = 1; ctx->last_buckets = B->n;
    if (reset_stats) CK(cudaMemsetAsync(ctx->stats, 0, sizeof(DevStats), st));
    if (B->n == 0) return PKDG_OK;
    if ((s = ensure(ctx, &ctx->desc, &ctx->desc_cap, B->n)) != PKDG_OK) return s;
    // the group kernel queues one entry per flagged SINK, the bucket kernel one per (bucket, pass)
    const int64_t fcap = G ? P->n + B->n + 16 : fix_capacity(B->n, P->n);
    if (!(flags & PKDG_NO_FIXUP) && (s = ensure(ctx, &ctx->fixq, &ctx->fixq_cap, fcap)) != PKDG_OK) return s;
    if (has_pc) {
        if ((s = ensure(ctx, &ctx->cellq, &ctx->cellq_cap, C->n * kCellQFloats)) != PKDG_OK) return s;
        if ((s = prep_cells(ctx, C, ctx->cellq, st)) != PKDG_OK) return s;
    }
    {
        int threads = 256;
        int64_t blocks = (B->n + threads - 1) / threads;
        const bool leaves = has_pp && (flags & PKDG_PP_LEAVES);
        if (leaves && (s = build_gfc(ctx, Bfull->first, Bfull->count, Bfull->n, P->n, st)) != PKDG_OK) return s;
        if (G) {   // buckets no group names get an empty descriptor
            CK(cudaMemsetAsync(ctx->desc, 0, sizeof(BucketDesc) * (size_t)B->n, st));
            const int64_t gblocks = (G->n + threads - 1) / threads;
            pkdg_pack_groups_kernel<<<(unsigned)(gblocks < 1 ? 1 : gblocks), threads, 0, st>>>(
                B->first, B->count, G->first_bucket, G->n_buckets, has_pp ? pp->offsets : nullptr,
                has_pc ? pc->offsets : nullptr, G->n, B->n, P->n, 0, 0, 0, ctx->desc, ctx->stats,
                ctx->counters + kMaxSlots, ctx->counters + 2 * kMaxSlots + 1, leaves ? pp->idx : nullptr, ctx->gfc,
                Bfull->n);
        } else {
            pkdg_pack_kernel<<<(unsigned)blocks, threads, 0, st>>>(B->first, B->count, has_pp ? pp->offsets : nullptr,
                                                                 has_pc ? pc->offsets : nullptr, B->n, P->n, 0, 0,
                                                                 ctx->desc, ctx->stats, ctx->counters + kMaxSlots,
                                                                 ctx->counters + 2 * kMaxSlots + 1,
                                                                 leaves ? pp->idx : nullptr, ctx->gfc, Bfull->n);
        }
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
    p.n_gbuckets = Bfull->n;
    p.cells_raw = has_pc ? C->rec : nullptr;
    p.cells_stride = has_pc ? C->stride_floats : PKDG_CELL_FLOATS;
    p.fix_queue = ctx->fixq;
    p.fix_count = ctx->counters + 2 * kMaxSlots + 1;
    p.fix_cap = (unsigned)(fcap > 0x7fffffffLL ? 0x7fffffffLL : fcap);
    if (G) { p.g_first = G->first_bucket; p.g_n = G->n_buckets; p.n_groups = G->n; p.g_base = 0; }
    if ((flags & PKDG_VALIDATE) && (s = launch_validate(ctx, p, true, st)) != PKDG_OK) return s;
    const bool prof = ctx->profiling && ctx->prof_n < 256;
    if (prof) {
        for (int i = 0; i < 3; ++i)
            if (!ctx->prof_ev[3 * ctx->prof_n + i]) CK(cudaEventCreate(&ctx->prof_ev[3 * ctx->prof_n + i]));
        CK(cudaEventRecord(ctx->prof_ev[3 * ctx->prof_n], st));
    }
    s = G ? launch_eval_groups(ctx, p, st) : launch_eval(ctx, p, st);
    if (prof) CK(cudaEventRecord(ctx->prof_ev[3 * ctx->prof_n + 1], st));
    if (s == PKDG_OK) s = launch_fixup(ctx, p, st);
    if (prof) {
        CK(cudaEventRecord(ctx->prof_ev[3 * ctx->prof_n + 2], st));
        ctx->prof_n++;
    }
    return s;
}

pkdg_status pkdg_gravity_eval(pkdg_ctx* ctx, const pkdg_particles* P, const pkdg_cells* C, const pkdg_buckets* B,
                              const pkdg_list* pp, const pkdg_list* pc, float eps, uint32_t flags, float* out,
                              void* stream) {
    return resident_impl(ctx, P, C, B, 0, B ? B->n : 0, nullptr, pp, pc, eps, flags, out, stream);
}

pkdg_status pkdg_gravity_eval_groups(pkdg_ctx* ctx, const pkdg_particles* P, const pkdg_cells* C, const pkdg_buckets* B,
                                     const pkdg_groups* G, const pkdg_list* pp, const pkdg_list* pc, float eps,
                                     uint32_t flags, float* out, void* stream) {
    if (!G) return fail(ctx, PKDG_EINVAL, "groups must not be NULL");
    return resident_impl(ctx, P, C, B, 0, B ? B->n : 0, G, pp, pc, eps, flags, out, stream);
}

pkdg_status pkdg_gravity_eval_range(pkdg_ctx* ctx, const pkdg_particles* P, const pkdg_cells* C, const pkdg_buckets* B,
                                    int64_t b0, int64_t b1, const pkdg_list* pp, const pkdg_list* pc, float eps,
                                    uint32_t flags, float* out, void* stream) {
    return resident_impl(ctx, P, C, B, b0, b1, nullptr, pp, pc, eps, flags, out, stream);
}

// ------------------------------------------------------------------------------------------------
// pkdg_gravity_eval_static: the resident call for hosts that cannot allocate (see include/pkdg.h).  Same four
// kernels as resident_impl, in the same order and with the same launch shapes, but no pkdg_ctx and no cudaMalloc /
// cudaFree anywhere below: all workspace pointers are offsets into g_static_scratch's device address.
// ------------------------------------------------------------------------------------------------
namespace {

constexpr int kStaticMaxDevices = 64;
struct StaticDev {
    bool ready = false;
    unsigned char* base = nullptr;   // DEVICE address of g_static_scratch on this device
    int num_sms = 0;
    int per_sm = 0;                  // CTAs per SM of the bucket kernel (particle lists)
};
StaticDev g_static_dev[kStaticMaxDevices];
std::mutex g_static_mu;              // guards g_static_dev (set-up may be raced by two host threads)

pkdg_status static_fail(pkdg_status s, const std::string& msg) {
    g_create_err = "pkdg_gravity_eval_static: " + msg;
    return s;
}

#define SCK(call)                                                                                  \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess) return static_fail(PKDG_ECUDA, std::string(#call) + ": " + cudaGetErrorString(e_)); \
    } while (0)

// Once per device, with that device current: where the array lives on THIS device, and what the launches need to
// know.  None of these calls allocates; they do reach the driver, hence "first call outside stream capture".
pkdg_status static_setup(int device, StaticDev** out) {
    std::lock_guard<std::mutex> lock(g_static_mu);
    StaticDev& d = g_static_dev[device];
    if (!d.ready) {
        unsigned char* base = nullptr;
        SCK(cudaGetSymbolAddress((void**)&base, g_static_scratch));
        if (!base || (reinterpret_cast<uintptr_t>(base) & 255u))
            return static_fail(PKDG_ECUDA, "cudaGetSymbolAddress gave no usable device address for the static workspace");
        int sms = 0, per_sm = 0;
        SCK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device));
        auto kern = pkdg_evalb_kernel<kBucketWarps, kBucketMinBlocks, false>;
        const int smem = kBucketWarps * (int)sizeof(WarpSmemB);
        SCK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        SCK(cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
        SCK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, kBucketWarps * 32, smem));
        d.base = base; d.num_sms = sms; d.per_sm = per_sm < 1 ? 1 : per_sm;
        d.ready = true;
    }
    *out = &d;
    return PKDG_OK;
}

}  // namespace

pkdg_status pkdg_gravity_eval_static(int device, const pkdg_particles* P, const pkdg_cells* C, const pkdg_buckets* B,
                                     const pkdg_list* pp, const pkdg_list* pc, float eps, uint32_t flags, float* out,
                                     void* stream) {
    // arguments and limits first: a refused call has touched neither the device nor the array
    if (device < 0 || device >= kStaticMaxDevices) return static_fail(PKDG_EINVAL, "device must be in 0..63");
    if (!P || !B || !out) return static_fail(PKDG_EINVAL, "particles, buckets and out must not be NULL");
    if (P->n < 0 || B->n < 0) return static_fail(PKDG_EINVAL, "negative size");
    if (flags & ~(uint32_t)(PKDG_ACCUMULATE | PKDG_SKIP_PP | PKDG_SKIP_PC | PKDG_NO_FIXUP | PKDG_FIXUP_ALL))
        return static_fail(PKDG_EINVAL, "only PKDG_ACCUMULATE, PKDG_SKIP_PP, PKDG_SKIP_PC, PKDG_NO_FIXUP and PKDG_FIXUP_ALL are "
                                        "supported (PKDG_PP_LEAVES and PKDG_VALIDATE need workspace this call does not have)");
    const bool has_pp = pp && pp->offsets;
    const bool pc_given = pc && pc->offsets;
    if (pc_given && (!C || C->n < 0 || (C->n > 0 && !C->rec) || C->stride_floats < PKDG_CELL_FLOATS))
        return static_fail(PKDG_EINVAL, "P-C list given without valid cells (stride_floats >= 36)");
    const int64_t nc = pc_given ? C->n : 0;
    if (B->n > PKDG_STATIC_MAX_BUCKETS || nc > PKDG_STATIC_MAX_CELLS || P->n > PKDG_STATIC_MAX_PARTICLES) {
        char msg[320];
        snprintf(msg, sizeof msg,
                 "problem too large for the static workspace: %lld buckets (limit %d), %lld cells (limit %d), %lld particles "
                 "(limit %d); split it into bucket ranges or use pkdg_gravity_eval with a context",
                 (long long)B->n, PKDG_STATIC_MAX_BUCKETS, (long long)nc, PKDG_STATIC_MAX_CELLS, (long long)P->n,
                 PKDG_STATIC_MAX_PARTICLES);
        return static_fail(PKDG_EINVAL, msg);
    }
    if (P->n > 0 && !P->xyzm) return static_fail(PKDG_EINVAL, "particles->xyzm is NULL");
    if (B->n > 0 && (!B->first || !B->count)) return static_fail(PKDG_EINVAL, "buckets->first/count is NULL");
    if (!aligned16(P->xyzm) || !aligned16(out)) return static_fail(PKDG_EINVAL, "xyzm and out must be 16-byte aligned");
    if (B->n == 0) return PKDG_OK;

    SCK(cudaSetDevice(device));
    StaticDev* d = nullptr;
    pkdg_status s = static_setup(device, &d);   // does work on the first call for this device only
    if (s != PKDG_OK) return s;
    cudaStream_t st = (cudaStream_t)stream;
    const bool has_pc = pc_given && nc > 0;

    DevStats* stats = reinterpret_cast<DevStats*>(d->base + kStOffStats);
    unsigned int* counters = reinterpret_cast<unsigned int*>(d->base + kStOffCounters);   // [0] work, [1] fix-up queue length
    BucketDesc* desc = reinterpret_cast<BucketDesc*>(d->base + kStOffDesc);
    float* cellq = reinterpret_cast<float*>(d->base + kStOffCellq);
    int4* fixq = reinterpret_cast<int4*>(d->base + kStOffFixq);

    // The array keeps the previous call's contents.  What has to start at zero is cleared here, in stream order ahead
    // of the kernels; descriptors [0, n_buckets), records [0, n_cells) and the queue entries below the queue length
    // are all written by this call before anything reads them.
    SCK(cudaMemsetAsync(stats, 0, sizeof(DevStats), st));
    SCK(cudaMemsetAsync(counters, 0, 2 * sizeof(unsigned int), st));
    if (has_pc) {
        const int64_t blocks = (nc + kPrepThreads - 1) / kPrepThreads;
        pkdg_prep_cells_kernel<<<(unsigned)blocks, kPrepThreads, 0, st>>>(C->rec, nc, C->stride_floats, cellq);
    }
    pkdg_pack_kernel<<<(unsigned)((B->n + 255) / 256), 256, 0, st>>>(
        B->first, B->count, has_pp ? pp->offsets : nullptr, has_pc ? pc->offsets : nullptr, B->n, P->n, 0, 0, desc, stats,
        counters, counters + 1, nullptr, nullptr, B->n);

    EvalParams p;
    p.xyzm = reinterpret_cast<const float4*>(P->xyzm);
    p.cellq = reinterpret_cast<const float4*>(cellq);
    p.desc = desc;
    p.pp_idx = has_pp ? pp->idx : nullptr;
    p.pc_idx = has_pc ? pc->idx : nullptr;
    p.gfc = nullptr;
    p.n_gbuckets = B->n;
    p.out = reinterpret_cast<float4*>(out);
    p.stats = stats;
    p.work_counter = counters;
    p.n_buckets = B->n; p.n_particles = P->n; p.n_cells = nc;
    const float h = 2.0f * eps;
    p.h2c = fmaxf(h * h, 1.0e-24f);
    p.eps = eps;
    p.flags = flags;
    p.cells_raw = has_pc ? C->rec : nullptr;
    p.cells_stride = has_pc ? C->stride_floats : PKDG_CELL_FLOATS;
    p.fix_k = (flags & PKDG_NO_FIXUP) ? -1.0f : (flags & PKDG_FIXUP_ALL) ? 0.0f : kDefaultKappa2 * kDefaultKappa2;
    p.fix_queue = fixq;
    p.fix_count = counters + 1;
    p.fix_cap = (unsigned)fix_capacity(B->n, P->n);   // <= kStFixCap by the limits above
    p.g_first = nullptr; p.g_n = nullptr; p.n_groups = 0; p.g_base = 0;

    {
        const int smem = kBucketWarps * (int)sizeof(WarpSmemB);
        int64_t grid = (int64_t)d->num_sms * d->per_sm;
        const int64_t want = (B->n + kBucketWarps - 1) / kBucketWarps;
        if (grid > want) grid = want;
        pkdg_evalb_kernel<kBucketWarps, kBucketMinBlocks, false><<<(unsigned)grid, kBucketWarps * 32, smem, st>>>(p);
    }
    if (p.fix_k >= 0.0f) {
        int64_t grid = B->n;
        const int64_t full = (int64_t)d->num_sms * 16;
        if (grid > full) grid = full;
        pkdg_fixup_kernel<<<(unsigned)grid, kFixThreads, 0, st>>>(p);
    }
    SCK(cudaGetLastError());
    return PKDG_OK;
}

// The FMM form of the path: the local expansion of every bucket from its C-C and C-P lists, evaluated at the
// bucket's particles (pkdg_fmm_kernel), then the P-P and P-C lists on top (PKDG_ACCUMULATE, so that the
// conditioning test of the evaluation kernel sees the total acceleration).
pkdg_status pkdg_gravity_eval_fmm(pkdg_ctx* ctx, const pkdg_particles* P, const pkdg_cells* C, const pkdg_buckets* B,
                                  const float* centres, const pkdg_list* pp, const pkdg_list* pc, const pkdg_list* cp,
                                  const pkdg_list* cc, float eps, uint32_t flags, float* out, void* stream) {
    pkdg_status s = check_common(ctx, P, C, B, pp, pc, out);
    if (s != PKDG_OK) return s;
    const bool has_cc = cc && cc->offsets, has_cp = cp && cp->offsets;
    const bool has_near = (pp && pp->offsets) || (pc && pc->offsets);
    if (has_cc) {
        if (!C || C->n < 0 || C->n > 0x7fffffffLL || (C->n > 0 && !C->rec) || C->stride_floats < PKDG_CELL_FLOATS)
            return fail(ctx, PKDG_EINVAL, "C-C list given without valid cells");
        if (!cc->idx && C->n > 0) return fail(ctx, PKDG_EINVAL, "cc->idx is NULL");
    }
    if (has_cp && !cp->idx && P->n > 0) return fail(ctx, PKDG_EINVAL, "cp->idx is NULL");
    if ((has_cc || has_cp) && B->n > 0 && !centres) return fail(ctx, PKDG_EINVAL, "centres must not be NULL with a C-C or C-P list");
    if (flags & PKDG_PP_LEAVES) return fail(ctx, PKDG_EINVAL, "PKDG_PP_LEAVES is not supported by pkdg_gravity_eval_fmm");
    cudaStream_t st = (cudaStream_t)stream;
    CK(cudaSetDevice(ctx->device));
    ctx->last_stream = st; ctx->last_chunks = 1; ctx->last_buckets = B->n;
    CK(cudaMemsetAsync(ctx->stats, 0, sizeof(DevStats), st));
    if (B->n == 0) return PKDG_OK;
    if (!has_cc && !has_cp) return resident_impl(ctx, P, C, B, 0, B->n, nullptr, pp, pc, eps, flags, out, stream, false);
    FmmParams f;
    f.xyzm = reinterpret_cast<const float4*>(P->xyzm);
    f.rec = has_cc ? C->rec : nullptr;
    f.stride = has_cc ? C->stride_floats : PKDG_CELL_FLOATS;
    f.rec_vec4 = has_cc && aligned16(C->rec) && (C->stride_floats % 4 == 0);
    f.n_particles = P->n; f.n_cells = has_cc ? C->n : 0; f.n_buckets = B->n;
    f.first = B->first; f.count = B->count; f.centre = centres;
    f.cc_off = has_cc ? cc->offsets : nullptr; f.cc_idx = has_cc ? cc->idx : nullptr;
    f.cp_off = has_cp ? cp->offsets : nullptr; f.cp_idx = has_cp ? cp->idx : nullptr;
    f.out = reinterpret_cast<float4*>(out);
    f.stats = ctx->stats;
    f.work_counter = ctx->counters + 2 * (kMaxSlots + 1);
    f.flags = flags;
    CK(cudaMemsetAsync(f.work_counter, 0, sizeof(unsigned int), st));
    int64_t grid = (int64_t)ctx->num_sms * 4;   // 128 registers: four CTAs of four warps per SM
    const int64_t want = (B->n + kFmmWarps - 1) / kFmmWarps;
    if (grid > want) grid = want;
    pkdg_fmm_kernel<<<(unsigned)grid, kFmmWarps * 32, 0, st>>>(f);
    ctx->launches++;
    CK(cudaGetLastError());
    if (!has_near) return PKDG_OK;
    return resident_impl(ctx, P, C, B, 0, B->n, nullptr, pp, pc, eps, flags | PKDG_ACCUMULATE, out, stream, false);
}

// out_host != NULL: the rows of every chunk (buckets are then known to be contiguous runs in ascending
// order, see pkdg_gravity_eval_host) are copied back on the chunk's stream right after its kernel, so
// the device->host traffic overlaps the host->device traffic of later chunks (PCIe is full duplex).
// Sinks are buckets [rb0, rb1) of Bfull (host arrays); the host lists hold rb1 - rb0 + 1 offsets.
// Gh != NULL (group-shared lists, host arrays): the unit of chunking is the group, the lists have Gh->n + 1
// offsets, the range must be all buckets and the groups must tile them in order.
static pkdg_status streamed_impl(pkdg_ctx* ctx, const pkdg_particles* P, const pkdg_cells* C,
                                 const pkdg_buckets* Bfull, int64_t rb0, int64_t rb1, const pkdg_groups* Gh,
                                 const pkdg_list* pph, const pkdg_list* pch, float eps, uint32_t flags, float* out,
                                 int32_t n_streams, int64_t max_entries, void* stream, float* out_host) {
    pkdg_status s = check_common(ctx, P, C, Bfull, pph, pch, out);
    if (s != PKDG_OK) return s;
    if (Gh) {
        if (Gh->n < 0 || (Gh->n > 0 && (!Gh->first_bucket || !Gh->n_buckets)))
            return fail(ctx, PKDG_EINVAL, "groups->first_bucket / n_buckets is NULL or n < 0");
        int64_t want = 0;
        for (int64_t g = 0; g < Gh->n; ++g) {
            if (Gh->first_bucket[g] != want || Gh->n_buckets[g] < 0)
                return fail(ctx, PKDG_EINVAL, "groups must tile the bucket range in order");
            want += Gh->n_buckets[g];
        }
        if (want != Bfull->n || rb0 != 0 || rb1 != Bfull->n)
            return fail(ctx, PKDG_EINVAL, "groups must tile the bucket range in order");
    }
    if (rb0 < 0 || rb1 < rb0 || rb1 > Bfull->n) return fail(ctx, PKDG_EINVAL, "bucket range outside [0, buckets->n]");
    const pkdg_buckets Bsub = {Bfull->first ? Bfull->first + rb0 : nullptr, Bfull->count ? Bfull->count + rb0 : nullptr,
                               rb1 - rb0};
    const pkdg_buckets* Bh = &Bsub;
    const int64_t nb_all = Bfull->n;
    if (n_streams < 1 || n_streams > kMaxSlots) return fail(ctx, PKDG_EINVAL, "n_streams must be in 1..8");
    if (max_entries < 1) return fail(ctx, PKDG_EINVAL, "max_entries_per_chunk must be >= 1");
    cudaStream_t st = (cudaStream_t)stream;
    CK(cudaSetDevice(ctx->device));
    const bool has_pp = pph && pph->offsets, has_pc = pch && pch->offsets && C && C->n > 0;
    const int64_t nb = Bh->n;
    ctx->last_stream = st; ctx->last_buckets = nb; ctx->last_chunks = 0;
    CK(cudaMemsetAsync(ctx->stats, 0, sizeof(DevStats), st));
    if (nb == 0) return PKDG_OK;
    const int64_t nu = Gh ? Gh->n : nb;   // units of chunking: groups or buckets
    if (nu == 0) return PKDG_OK;
    if ((s = ensure_slots(ctx, n_streams)) != PKDG_OK) return s;
    if (has_pc) {
        if ((s = ensure(ctx, &ctx->cellq, &ctx->cellq_cap, C->n * kCellQFloats)) != PKDG_OK) return s;
        if ((s = prep_cells(ctx, C, ctx->cellq, st)) != PKDG_OK) return s;
    }
    const bool leaves = has_pp && (flags & PKDG_PP_LEAVES);
    if (leaves) {  // leaf references may point at any bucket: all (first, count) pairs go to the device first
        if ((s = ensure(ctx, &ctx->g_first, &ctx->g_first_cap, nb_all)) != PKDG_OK) return s;
        if ((s = ensure(ctx, &ctx->g_count, &ctx->g_count_cap, nb_all)) != PKDG_OK) return s;
        CK(cudaMemcpyAsync(ctx->g_first, Bfull->first, sizeof(int32_t) * nb_all, cudaMemcpyHostToDevice, st));
        CK(cudaMemcpyAsync(ctx->g_count, Bfull->count, sizeof(int32_t) * nb_all, cudaMemcpyHostToDevice, st));
        if ((s = build_gfc(ctx, ctx->g_first, ctx->g_count, nb_all, P->n, st)) != PKDG_OK) return s;
    }
    CK(cudaEventRecord(ctx->ev_ready, st));
    int64_t* bounds = (int64_t*)malloc(sizeof(int64_t) * (size_t)(nu + 1));
    if (!bounds) return fail(ctx, PKDG_ENOMEM, "host malloc of chunk bounds failed");
    const int64_t nchunk = chunk_bounds_host(nu, has_pp ? pph->offsets : nullptr, has_pc ? pch->offsets : nullptr,
                                             max_entries, bounds);
    ctx->last_chunks = nchunk;
    pkdg_status rc = PKDG_OK;
    for (int i = 0; i < n_streams; ++i) {
        if (cudaStreamWaitEvent(ctx->slots[i].st, ctx->ev_ready, 0) != cudaSuccess) rc = PKDG_ECUDA;
        ctx->slots[i].busy = false;
    }
    for (int64_t ic = 0; ic < nchunk && rc == PKDG_OK; ++ic) {
        Slot& sl = ctx->slots[ic % n_streams];
        const int64_t u0 = bounds[ic], u1 = bounds[ic + 1], cu = u1 - u0;   // units, then their buckets
        const int64_t b0 = Gh ? Gh->first_bucket[u0] : u0;
        const int64_t b1 = Gh ? (int64_t)Gh->first_bucket[u1 - 1] + Gh->n_buckets[u1 - 1] : u1, cb = b1 - b0;
        const int64_t pbase = has_pp ? pph->offsets[u0] : 0, plen = has_pp ? pph->offsets[u1] - pbase : 0;
        const int64_t cbase = has_pc ? pch->offsets[u0] : 0, clen = has_pc ? pch->offsets[u1] - cbase : 0;
        // bounded in-flight work: a slot is reused only after its previous chunk is done
        if (sl.busy && cudaEventSynchronize(sl.done) != cudaSuccess) { rc = PKDG_ECUDA; break; }
        if ((rc = ensure(ctx, &sl.pp_idx, &sl.cap_pp, plen)) != PKDG_OK) break;
        if ((rc = ensure(ctx, &sl.pc_idx, &sl.cap_pc, clen)) != PKDG_OK) break;
        int64_t chunk_sinks = 0;
        for (int64_t b = b0; b < b1; ++b) chunk_sinks += Bh->count[b] > 0 ? Bh->count[b] : 0;
        const int64_t fcap = Gh ? chunk_sinks + cb + 16 : fix_capacity(cb, chunk_sinks);
        if (!(flags & PKDG_NO_FIXUP) && (rc = ensure(ctx, &sl.fixq, &sl.fixq_cap, fcap)) != PKDG_OK) break;
        if (cb + 1 > sl.cap_b) {
            int64_t c1 = 0, c2 = 0, c5 = 0;
            cudaFree(sl.first); cudaFree(sl.count); cudaFree(sl.desc);
            sl.first = sl.count = nullptr; sl.desc = nullptr; sl.cap_b = 0;
            if ((rc = ensure(ctx, &sl.first, &c1, cb + 1)) != PKDG_OK) break;
            if ((rc = ensure(ctx, &sl.count, &c2, cb + 1)) != PKDG_OK) break;
            if ((rc = ensure(ctx, &sl.desc, &c5, cb + 1)) != PKDG_OK) break;
            sl.cap_b = c1;
        }
        if (cu + 1 > sl.cap_off) {
            int64_t c3 = 0, c4 = 0;
            cudaFree(sl.pp_off); cudaFree(sl.pc_off);
            sl.pp_off = sl.pc_off = nullptr; sl.cap_off = 0;
            if ((rc = ensure(ctx, &sl.pp_off, &c3, cu + 1)) != PKDG_OK) break;
            if ((rc = ensure(ctx, &sl.pc_off, &c4, cu + 1)) != PKDG_OK) break;
            sl.cap_off = c3;
        }
        if (Gh && cu > sl.cap_g) {
            int64_t c6 = 0, c7 = 0;
            cudaFree(sl.gfirst); cudaFree(sl.gn);
            sl.gfirst = sl.gn = nullptr; sl.cap_g = 0;
            if ((rc = ensure(ctx, &sl.gfirst, &c6, cu)) != PKDG_OK) break;
            if ((rc = ensure(ctx, &sl.gn, &c7, cu)) != PKDG_OK) break;
            sl.cap_g = c6;
        }
        cudaError_t e = cudaMemcpyAsync(sl.first, Bh->first + b0, sizeof(int32_t) * cb, cudaMemcpyHostToDevice, sl.st);
        if (e == cudaSuccess) e = cudaMemcpyAsync(sl.count, Bh->count + b0, sizeof(int32_t) * cb, cudaMemcpyHostToDevice, sl.st);
        if (e == cudaSuccess && Gh) {
            e = cudaMemcpyAsync(sl.gfirst, Gh->first_bucket + u0, sizeof(int32_t) * cu, cudaMemcpyHostToDevice, sl.st);
            if (e == cudaSuccess) e = cudaMemcpyAsync(sl.gn, Gh->n_buckets + u0, sizeof(int32_t) * cu, cudaMemcpyHostToDevice, sl.st);
        }
        if (e == cudaSuccess && has_pp) {
            e = cudaMemcpyAsync(sl.pp_off, pph->offsets + u0, sizeof(int64_t) * (cu + 1), cudaMemcpyHostToDevice, sl.st);
            if (e == cudaSuccess && plen)
                e = cudaMemcpyAsync(sl.pp_idx, pph->idx + pbase, sizeof(int32_t) * plen, cudaMemcpyHostToDevice, sl.st);
        }
        if (e == cudaSuccess && has_pc) {
            e = cudaMemcpyAsync(sl.pc_off, pch->offsets + u0, sizeof(int64_t) * (cu + 1), cudaMemcpyHostToDevice, sl.st);
            if (e == cudaSuccess && clen)
                e = cudaMemcpyAsync(sl.pc_idx, pch->idx + cbase, sizeof(int32_t) * clen, cudaMemcpyHostToDevice, sl.st);
        }
        if (e != cudaSuccess) { rc = fail(ctx, PKDG_ECUDA, std::string("chunk copy: ") + cudaGetErrorString(e)); break; }
        unsigned int* counter = ctx->counters + (ic % n_streams);
        int threads = 256;
        if (Gh) {
            pkdg_pack_groups_kernel<<<(unsigned)((cu + threads - 1) / threads), threads, 0, sl.st>>>(
                sl.first, sl.count, sl.gfirst, sl.gn, has_pp ? sl.pp_off : nullptr, has_pc ? sl.pc_off : nullptr, cu, cb,
                P->n, pbase, cbase, b0, sl.desc, ctx->stats, counter, counter + kMaxSlots + 1,
                leaves ? sl.pp_idx : nullptr, ctx->gfc, nb_all);
        } else {
            pkdg_pack_kernel<<<(unsigned)((cb + threads - 1) / threads), threads, 0, sl.st>>>(
                sl.first, sl.count, has_pp ? sl.pp_off : nullptr, has_pc ? sl.pc_off : nullptr, cb, P->n, pbase, cbase,
                sl.desc, ctx->stats, counter, counter + kMaxSlots + 1, leaves ? sl.pp_idx : nullptr, ctx->gfc, nb_all);
        }
        ctx->launches++;
        EvalParams p;
        fill_params(p, ctx, P->xyzm, P->n, has_pc ? C->n : 0, eps, flags, out);
        p.desc = sl.desc;
        p.pp_idx = sl.pp_idx;
        p.pc_idx = sl.pc_idx;
        p.work_counter = counter;
        p.n_buckets = cb;
        p.gfc = ctx->gfc;
        p.n_gbuckets = nb_all;
        p.cells_raw = has_pc ? C->rec : nullptr;
        p.cells_stride = has_pc ? C->stride_floats : PKDG_CELL_FLOATS;
        p.fix_queue = sl.fixq;
        p.fix_count = counter + kMaxSlots + 1;
        p.fix_cap = (unsigned)(fcap > 0x7fffffffLL ? 0x7fffffffLL : fcap);
        if (Gh) { p.g_first = sl.gfirst; p.g_n = sl.gn; p.n_groups = cu; p.g_base = b0; }
        if ((flags & PKDG_VALIDATE) && (rc = launch_validate(ctx, p, ic == 0, sl.st)) != PKDG_OK) break;
        if ((rc = Gh ? launch_eval_groups(ctx, p, sl.st) : launch_eval(ctx, p, sl.st)) != PKDG_OK) break;
        if ((rc = launch_fixup(ctx, p, sl.st)) != PKDG_OK) break;
        if (out_host && cb > 0) {
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
    return streamed_impl(ctx, P, C, Bh, 0, Bh ? Bh->n : 0, nullptr, pph, pch, eps, flags, out, n_streams, max_entries,
                         stream, nullptr);
}

static pkdg_status host_impl(pkdg_ctx* ctx, const pkdg_particles* Ph, const pkdg_cells* Ch, const pkdg_buckets* Bfull,
                             int64_t rb0, int64_t rb1, const pkdg_groups* Gh, const pkdg_list* pph, const pkdg_list* pch,
                             float eps, uint32_t flags, float* out_host, int32_t n_streams, int64_t max_entries) {
    pkdg_status s = check_common(ctx, Ph, Ch, Bfull, pph, pch, out_host);
    if (s != PKDG_OK) return s;
    if (rb0 < 0 || rb1 < rb0 || rb1 > Bfull->n) return fail(ctx, PKDG_EINVAL, "bucket range outside [0, buckets->n]");
    const pkdg_buckets Bsub = {Bfull->first ? Bfull->first + rb0 : nullptr, Bfull->count ? Bfull->count + rb0 : nullptr,
                               rb1 - rb0};
    const pkdg_buckets* Bh = &Bsub;
    CK(cudaSetDevice(ctx->device));
    if (!ctx->own_stream) CK(cudaStreamCreateWithFlags(&ctx->own_stream, cudaStreamNonBlocking));
    cudaStream_t st = ctx->own_stream;
    const bool has_pc = pch && pch->offsets && Ch && Ch->n > 0;
    // all workspace first: nothing may fail between the first copy out of the caller's buffers and the
    // synchronisation at the bottom except inside `run`, whose every way out passes that synchronisation
    if ((s = ensure(ctx, &ctx->e2e_xyzm, &ctx->e2e_np, Ph->n * 4)) != PKDG_OK) return s;
    if ((s = ensure(ctx, &ctx->e2e_out, &ctx->e2e_no, Ph->n * 4)) != PKDG_OK) return s;
    if (has_pc && (s = ensure(ctx, &ctx->e2e_cells, &ctx->e2e_nc, Ch->n * (int64_t)Ch->stride_floats)) != PKDG_OK) return s;
    auto run = [&]() -> pkdg_status {
        pkdg_status s = PKDG_OK;
        if (Ph->n) CK(cudaMemcpyAsync(ctx->e2e_xyzm, Ph->xyzm, sizeof(float) * 4 * Ph->n, cudaMemcpyHostToDevice, st));
        pkdg_cells Cd = {nullptr, 0, PKDG_CELL_FLOATS};
        if (has_pc) {
            CK(cudaMemcpyAsync(ctx->e2e_cells, Ch->rec, sizeof(float) * Ch->n * Ch->stride_floats, cudaMemcpyHostToDevice, st));
            Cd.rec = ctx->e2e_cells; Cd.n = Ch->n; Cd.stride_floats = Ch->stride_floats;
        }
        // tree-ordered sinks (every bucket of the range starts where the previous one ends: the rows form one run):
        // each chunk's rows go back as soon as they are done and nothing else is copied.  Anything else: the caller's
        // rows make a round trip, so that rows in no listed bucket keep their values.
        bool one_run = Bh->n > 0;
        for (int64_t b = 0; one_run && b < Bh->n; ++b) {
            const int64_t end = (int64_t)Bh->first[b] + Bh->count[b];
            one_run = Bh->count[b] >= 0 && Bh->first[b] >= 0 && end <= Ph->n && (b + 1 == Bh->n || end == (int64_t)Bh->first[b + 1]);
        }
        if (Ph->n && (!one_run || (flags & PKDG_ACCUMULATE))) {
            int64_t r0 = 0, r1 = Ph->n;
            if (one_run) { r0 = Bh->first[0]; r1 = (int64_t)Bh->first[Bh->n - 1] + Bh->count[Bh->n - 1]; }
            if (r1 > r0)
                CK(cudaMemcpyAsync(ctx->e2e_out + 4 * r0, out_host + 4 * r0, sizeof(float) * 4 * (size_t)(r1 - r0),
                                   cudaMemcpyHostToDevice, st));
        }
        pkdg_particles Pd = {ctx->e2e_xyzm, Ph->n};
        s = streamed_impl(ctx, &Pd, has_pc ? &Cd : nullptr, Bfull, rb0, rb1, Gh, pph, has_pc ? pch : nullptr, eps, flags,
                          ctx->e2e_out, n_streams, max_entries, st, one_run ? out_host : nullptr);
        if (s == PKDG_OK && !one_run && Ph->n) {
            cudaError_t e = cudaMemcpyAsync(out_host, ctx->e2e_out, sizeof(float) * 4 * Ph->n, cudaMemcpyDeviceToHost, st);
            if (e != cudaSuccess) s = fail(ctx, PKDG_ECUDA, cudaGetErrorString(e));
        }
        return s;
    };
    s = run();
    // also on the error path: no copy that touches the caller's host buffers may still be in flight on return
    for (int i = 0; i < ctx->n_slots_live; ++i) cudaStreamSynchronize(ctx->slots[i].st);
    cudaError_t e = cudaStreamSynchronize(st);
    if (s == PKDG_OK && e != cudaSuccess) s = fail(ctx, PKDG_ECUDA, cudaGetErrorString(e));
    return s;
}

pkdg_status pkdg_gravity_eval_host_range(pkdg_ctx* ctx, const pkdg_particles* Ph, const pkdg_cells* Ch,
                                         const pkdg_buckets* Bfull, int64_t rb0, int64_t rb1, const pkdg_list* pph,
                                         const pkdg_list* pch, float eps, uint32_t flags, float* out_host,
                                         int32_t n_streams, int64_t max_entries) {
    return host_impl(ctx, Ph, Ch, Bfull, rb0, rb1, nullptr, pph, pch, eps, flags, out_host, n_streams, max_entries);
}

pkdg_status pkdg_gravity_eval_host(pkdg_ctx* ctx, const pkdg_particles* Ph, const pkdg_cells* Ch,
                                   const pkdg_buckets* Bh, const pkdg_list* pph, const pkdg_list* pch, float eps,
                                   uint32_t flags, float* out_host, int32_t n_streams, int64_t max_entries) {
    return host_impl(ctx, Ph, Ch, Bh, 0, Bh ? Bh->n : 0, nullptr, pph, pch, eps, flags, out_host, n_streams, max_entries);
}

pkdg_status pkdg_gravity_eval_host_groups(pkdg_ctx* ctx, const pkdg_particles* Ph, const pkdg_cells* Ch,
                                          const pkdg_buckets* Bh, const pkdg_groups* Gh, const pkdg_list* pph,
                                          const pkdg_list* pch, float eps, uint32_t flags, float* out_host,
                                          int32_t n_streams, int64_t max_entries) {
    if (!Gh) return fail(ctx, PKDG_EINVAL, "groups must not be NULL");
    return host_impl(ctx, Ph, Ch, Bh, 0, Bh ? Bh->n : 0, Gh, pph, pch, eps, flags, out_host, n_streams, max_entries);
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

// Exclusive scan of v[0 .. n) in place, total at v[n] (device).
static pkdg_status device_scan(pkdg_ctx* ctx, int64_t* v, int64_t n, cudaStream_t st) {
    const int64_t per = (int64_t)kScanBlock * kScanItems;
    const int64_t nblk = n > 0 ? (n + per - 1) / per : 1;
    pkdg_status s = ensure(ctx, &ctx->scan_tmp, &ctx->scan_cap, nblk + 1);
    if (s != PKDG_OK) return s;
    pkdg_scan_blocks_kernel<<<(unsigned)nblk, kScanBlock, 0, st>>>(v, n, ctx->scan_tmp);
    pkdg_scan_kernel<<<1, 1024, 0, st>>>(ctx->scan_tmp, nblk);
    pkdg_scan_add_kernel<<<(unsigned)((n + 1 + 255) / 256), 256, 0, st>>>(v, n, ctx->scan_tmp, nblk);
    ctx->launches += 3;
    CK(cudaGetLastError());
    return PKDG_OK;
}

static pkdg_status check_tree(pkdg_ctx* ctx, const pkdg_tree* T, const pkdg_cells* C, const int32_t* sink_cell,
                              int64_t n_sinks, double theta) {
    if (!ctx) return PKDG_EINVAL;
    if (!T || !C || !T->first || !T->count || !T->end || !T->isleaf || !T->bblo || !T->bbhi || !C->rec)
        return fail(ctx, PKDG_EINVAL, "tree arrays and cell records must not be NULL");
    if (T->n_cells < 0 || T->n_cells != C->n || C->stride_floats < PKDG_CELL_FLOATS || T->n_cells > 0x7fffffffLL)
        return fail(ctx, PKDG_EINVAL, "tree->n_cells must equal cells->n; stride_floats >= 36");
    if (n_sinks < 0 || (n_sinks > 0 && !sink_cell)) return fail(ctx, PKDG_EINVAL, "sink_cell is NULL or n_sinks < 0");
    if (!(theta > 0.0)) return fail(ctx, PKDG_EINVAL, "theta must be > 0");
    return PKDG_OK;
}

static TreeView tree_view(const pkdg_tree* T, const pkdg_cells* C, bool leaves) {
    TreeView v;
    v.first = T->first; v.count = T->count; v.end = T->end; v.isleaf = T->isleaf;
    v.bblo = T->bblo; v.bbhi = T->bbhi; v.rec = C->rec; v.stride = C->stride_floats; v.n_cells = T->n_cells;
    v.leaf_rank = leaves ? T->leaf_rank : nullptr;
    return v;
}

// the walk's 64-byte cell records (workspace of the context)
static pkdg_status walk_nodes(pkdg_ctx* ctx, const TreeView& v, double theta, cudaStream_t st, bool count_bad) {
    pkdg_status s = ensure(ctx, &ctx->wnodes, &ctx->wnodes_cap, v.n_cells);
    if (s != PKDG_OK || v.n_cells == 0) return s;
    pkdg_walk_nodes_kernel<<<(unsigned)((v.n_cells + 255) / 256), 256, 0, st>>>(v, theta, ctx->wnodes,
                                                                               count_bad ? ctx->stats : nullptr);
    ctx->launches++;
    CK(cudaGetLastError());
    return PKDG_OK;
}

pkdg_status pkdg_build_lists_count(pkdg_ctx* ctx, const pkdg_tree* T, const pkdg_cells* C, const int32_t* sink_cell,
                                   int64_t n_sinks, double theta, double eps, uint32_t flags, int64_t* pp_off,
                                   int64_t* pc_off, int64_t* totals_host, void* stream) {
    pkdg_status s = check_tree(ctx, T, C, sink_cell, n_sinks, theta);
    if (s != PKDG_OK) return s;
    if (!pp_off || !pc_off) return fail(ctx, PKDG_EINVAL, "pp_offsets / pc_offsets must not be NULL");
    if ((flags & PKDG_PP_LEAVES) && !T->leaf_rank) return fail(ctx, PKDG_EINVAL, "PKDG_PP_LEAVES needs tree->leaf_rank");
    cudaStream_t st = (cudaStream_t)stream;
    CK(cudaSetDevice(ctx->device));
    const TreeView v = tree_view(T, C, (flags & PKDG_PP_LEAVES) != 0);
    // malformed tree input (a subtree end that does not advance, a sink that is no cell of the tree) is counted in
    // bad_entries: pkdg_get_stats after this call reports it (an evaluation call resets the counters)
    ctx->last_stream = st; ctx->last_chunks = 1; ctx->last_buckets = n_sinks;
    CK(cudaMemsetAsync(ctx->stats, 0, sizeof(DevStats), st));
    if ((s = walk_nodes(ctx, v, theta, st, true)) != PKDG_OK) return s;
    if (n_sinks > 0) {
        pkdg_walk_kernel<false><<<(unsigned)((n_sinks + 127) / 128), 128, 0, st>>>(
            ctx->wnodes, v.n_cells, (flags & PKDG_PP_LEAVES) != 0, sink_cell, n_sinks, theta, eps, pp_off, pc_off, nullptr,
            nullptr, nullptr, nullptr, ctx->stats);
        ctx->launches++;
        CK(cudaGetLastError());
    }
    if ((s = device_scan(ctx, pp_off, n_sinks, st)) != PKDG_OK) return s;
    if ((s = device_scan(ctx, pc_off, n_sinks, st)) != PKDG_OK) return s;
    if (totals_host) {   // the caller allocates the index arrays from these: synchronous
        CK(cudaMemcpyAsync(totals_host, pp_off + n_sinks, sizeof(int64_t), cudaMemcpyDeviceToHost, st));
        CK(cudaMemcpyAsync(totals_host + 1, pc_off + n_sinks, sizeof(int64_t), cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
    }
    return PKDG_OK;
}

pkdg_status pkdg_build_lists_fill(pkdg_ctx* ctx, const pkdg_tree* T, const pkdg_cells* C, const int32_t* sink_cell,
                                  int64_t n_sinks, double theta, double eps, uint32_t flags, const int64_t* pp_off,
                                  const int64_t* pc_off, int32_t* pp_idx, int32_t* pc_idx, void* stream) {
    pkdg_status s = check_tree(ctx, T, C, sink_cell, n_sinks, theta);
    if (s != PKDG_OK) return s;
    if (!pp_off || !pc_off) return fail(ctx, PKDG_EINVAL, "pp_offsets / pc_offsets must not be NULL");
    if ((flags & PKDG_PP_LEAVES) && !T->leaf_rank) return fail(ctx, PKDG_EINVAL, "PKDG_PP_LEAVES needs tree->leaf_rank");
    if (n_sinks == 0) return PKDG_OK;
    cudaStream_t st = (cudaStream_t)stream;
    CK(cudaSetDevice(ctx->device));
    const TreeView v = tree_view(T, C, (flags & PKDG_PP_LEAVES) != 0);
    if ((s = walk_nodes(ctx, v, theta, st, false)) != PKDG_OK) return s;   // rebuilt here: the caller may have changed the tree since _count
    pkdg_walk_kernel<true><<<(unsigned)((n_sinks + 127) / 128), 128, 0, st>>>(
        ctx->wnodes, v.n_cells, (flags & PKDG_PP_LEAVES) != 0, sink_cell, n_sinks, theta, eps, nullptr, nullptr, pp_off,
        pc_off, pp_idx, pc_idx, nullptr);
    ctx->launches++;
    CK(cudaGetLastError());
    return PKDG_OK;
}

// End to end from the TREE: every buffer on the host, lists built on the device.  Tree, cells and buckets go first;
// the walk runs while the particles are still crossing the bus; the evaluation is cut into n_ranges bucket ranges and
// the rows of a range go back while the next range is evaluated.
pkdg_status pkdg_gravity_eval_tree_host(pkdg_ctx* ctx, const pkdg_particles* Ph, const pkdg_cells* Ch, const pkdg_tree* Th,
                                        const pkdg_buckets* Bh, const int32_t* bucket_cell_host, double theta, float eps,
                                        uint32_t flags, float* out_host, int32_t n_ranges) {
    if (!ctx) return PKDG_EINVAL;
    if (!Ph || !Ch || !Th || !Bh || !out_host) return fail(ctx, PKDG_EINVAL, "particles, cells, tree, buckets and out must not be NULL");
    pkdg_status s = check_tree(ctx, Th, Ch, bucket_cell_host, Bh->n, theta);
    if (s != PKDG_OK) return s;
    if ((s = check_common(ctx, Ph, Ch, Bh, nullptr, nullptr, out_host)) != PKDG_OK) return s;
    if (n_ranges < 1 || n_ranges > 64) return fail(ctx, PKDG_EINVAL, "n_ranges must be in 1..64");
    if (flags & (PKDG_ACCUMULATE | PKDG_SKIP_PP | PKDG_SKIP_PC))
        return fail(ctx, PKDG_EINVAL, "pkdg_gravity_eval_tree_host takes PKDG_NO_FIXUP, PKDG_FIXUP_ALL and PKDG_VALIDATE only");
    const int64_t nb = Bh->n, ncell = Th->n_cells, np = Ph->n;
    for (int64_t b = 0; b < nb; ++b) {   // rows go back range by range: the buckets must be the contiguous runs of tree order
        const int64_t end = (int64_t)Bh->first[b] + Bh->count[b];
        if (Bh->count[b] < 0 || Bh->first[b] < 0 || end > np || (b + 1 < nb && end != (int64_t)Bh->first[b + 1]) ||
            bucket_cell_host[b] < 0 || bucket_cell_host[b] >= ncell)
            return fail(ctx, PKDG_EINVAL, "buckets must be contiguous runs in ascending order and name cells of the tree");
        const int32_t c = bucket_cell_host[b];
        if (!Th->isleaf[c] || Th->first[c] != Bh->first[b] || Th->count[c] != Bh->count[b])
            return fail(ctx, PKDG_EINVAL, "bucket_cell_host[b] must be a leaf cell whose particle run is bucket b");
    }
    for (int64_t k = 0; k < ncell; ++k)   // the walk advances through end[]: it must move forward and stay inside
        if (Th->end[k] <= k || Th->end[k] > ncell)
            return fail(ctx, PKDG_EINVAL, "tree_host->end[k] must lie in (k, n_cells]");
    // The walk names a P-P source leaf by its bucket index, so EVERY leaf must be a bucket.  The leaves partition the
    // root's particle run; contiguous leaf runs that start and end where the root does are therefore all of them.
    if (nb > 0 && ncell > 0) {
        const int64_t r0 = Th->first[0], r1 = (int64_t)Th->first[0] + Th->count[0];
        if ((int64_t)Bh->first[0] != r0 || (int64_t)Bh->first[nb - 1] + Bh->count[nb - 1] != r1)
            return fail(ctx, PKDG_EINVAL, "buckets_host must be ALL leaves of the tree (a subset of sinks is not supported: "
                                          "use pkdg_build_lists_* and pkdg_gravity_eval_range)");
    }
    CK(cudaSetDevice(ctx->device));
    if (!ctx->own_stream) CK(cudaStreamCreateWithFlags(&ctx->own_stream, cudaStreamNonBlocking));
    if ((s = ensure_slots(ctx, 1)) != PKDG_OK) return s;
    for (cudaEvent_t& e : ctx->t_ev)
        if (!e) CK(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    cudaStream_t sa = ctx->own_stream, sb = ctx->slots[0].st;
    if (nb == 0 || np == 0) return PKDG_OK;
    // everything that queues work runs in this lambda, so that every way out of it passes the synchronisation below:
    // no copy that touches the caller's host buffers may still be in flight when the call returns
    auto run = [&]() -> pkdg_status {
        pkdg_status s = PKDG_OK;
        // workspace
        if ((s = ensure(ctx, &ctx->e2e_xyzm, &ctx->e2e_np, np * 4)) != PKDG_OK) return s;
        if ((s = ensure(ctx, &ctx->e2e_out, &ctx->e2e_no, np * 4)) != PKDG_OK) return s;
        if ((s = ensure(ctx, &ctx->e2e_cells, &ctx->e2e_nc, ncell * (int64_t)Ch->stride_floats)) != PKDG_OK) return s;
        if ((s = ensure(ctx, &ctx->t_first, &ctx->t_cap[0], ncell)) != PKDG_OK) return s;
        if ((s = ensure(ctx, &ctx->t_count, &ctx->t_cap[1], ncell)) != PKDG_OK) return s;
        if ((s = ensure(ctx, &ctx->t_end, &ctx->t_cap[2], ncell)) != PKDG_OK) return s;
        if ((s = ensure(ctx, &ctx->t_isleaf, &ctx->t_cap[3], ncell)) != PKDG_OK) return s;
        if ((s = ensure(ctx, &ctx->t_rank, &ctx->t_cap[4], ncell)) != PKDG_OK) return s;
        if ((s = ensure(ctx, &ctx->t_sink, &ctx->t_cap[5], nb)) != PKDG_OK) return s;
        if ((s = ensure(ctx, &ctx->t_bblo, &ctx->t_cap[6], 3 * ncell)) != PKDG_OK) return s;
        if ((s = ensure(ctx, &ctx->t_bbhi, &ctx->t_cap[7], 3 * ncell)) != PKDG_OK) return s;
        if ((s = ensure(ctx, &ctx->t_bfirst, &ctx->t_bcap[0], nb)) != PKDG_OK) return s;
        if ((s = ensure(ctx, &ctx->t_bcount, &ctx->t_bcap[1], nb)) != PKDG_OK) return s;
        if ((s = ensure(ctx, &ctx->t_ppo, &ctx->t_bcap[2], nb + 1)) != PKDG_OK) return s;
        if ((s = ensure(ctx, &ctx->t_pco, &ctx->t_bcap[3], nb + 1)) != PKDG_OK) return s;
        // tree, cells, buckets on stream a; particles on stream b
        auto h2d = [&](void* d, const void* h, size_t bytes, cudaStream_t st) { return cudaMemcpyAsync(d, h, bytes, cudaMemcpyHostToDevice, st); };
        CK(h2d(ctx->e2e_cells, Ch->rec, sizeof(float) * ncell * Ch->stride_floats, sa));
        CK(h2d(ctx->t_first, Th->first, 4 * ncell, sa)); CK(h2d(ctx->t_count, Th->count, 4 * ncell, sa));
        CK(h2d(ctx->t_end, Th->end, 4 * ncell, sa)); CK(h2d(ctx->t_isleaf, Th->isleaf, 4 * ncell, sa));
        CK(h2d(ctx->t_bblo, Th->bblo, 12 * ncell, sa)); CK(h2d(ctx->t_bbhi, Th->bbhi, 12 * ncell, sa));
        CK(h2d(ctx->t_sink, bucket_cell_host, 4 * nb, sa));
        CK(h2d(ctx->t_bfirst, Bh->first, 4 * nb, sa)); CK(h2d(ctx->t_bcount, Bh->count, 4 * nb, sa));
        CK(h2d(ctx->e2e_xyzm, Ph->xyzm, sizeof(float) * 4 * np, sb));
        CK(cudaEventRecord(ctx->t_ev[0], sb));
        // leaf_rank[cell of bucket b] = b, then the walk (P-P entries as bucket references).  A cell no bucket names
        // keeps 0x7f7f7f7f, which the packer counts as a bad entry (it cannot happen after the checks above).
        CK(cudaMemsetAsync(ctx->t_rank, 0x7f, sizeof(int32_t) * (size_t)ncell, sa));
        pkdg_leaf_rank_kernel<<<(unsigned)((nb + 255) / 256), 256, 0, sa>>>(ctx->t_sink, nb, ctx->t_rank);
        ctx->launches++;
        pkdg_tree Td = {ctx->t_first, ctx->t_count, ctx->t_end, ctx->t_isleaf, ctx->t_bblo, ctx->t_bbhi, ctx->t_rank, ncell};
        pkdg_cells Cd = {ctx->e2e_cells, ncell, Ch->stride_floats};
        int64_t tot[2] = {0, 0};
        if ((s = pkdg_build_lists_count(ctx, &Td, &Cd, ctx->t_sink, nb, theta, (double)eps, PKDG_PP_LEAVES, ctx->t_ppo, ctx->t_pco,
                                        tot, sa)) != PKDG_OK) return s;
        if ((s = ensure(ctx, &ctx->t_ppi, &ctx->t_bcap[4], tot[0] + 1)) != PKDG_OK) return s;
        if ((s = ensure(ctx, &ctx->t_pci, &ctx->t_bcap[5], tot[1] + 1)) != PKDG_OK) return s;
        if ((s = pkdg_build_lists_fill(ctx, &Td, &Cd, ctx->t_sink, nb, theta, (double)eps, PKDG_PP_LEAVES, ctx->t_ppo, ctx->t_pco,
                                       ctx->t_ppi, ctx->t_pci, sa)) != PKDG_OK) return s;
        CK(cudaStreamWaitEvent(sa, ctx->t_ev[0], 0));
        // evaluation in bucket ranges; rows of a range go back on stream b while the next range runs
        pkdg_particles Pd = {ctx->e2e_xyzm, np};
        pkdg_buckets Bd = {ctx->t_bfirst, ctx->t_bcount, nb};
        pkdg_status rc = PKDG_OK;
        bool first_range = true;
        for (int r = 0; r < n_ranges && rc == PKDG_OK; ++r) {
            const int64_t b0 = nb * r / n_ranges, b1 = nb * (r + 1) / n_ranges;
            if (b1 <= b0) continue;
            pkdg_list pp = {ctx->t_ppo + b0, ctx->t_ppi}, pc = {ctx->t_pco + b0, ctx->t_pci};
            // the counters are reset by the first range only: they add up over the call
            rc = resident_impl(ctx, &Pd, &Cd, &Bd, b0, b1, nullptr, &pp, &pc, eps, flags | PKDG_PP_LEAVES, ctx->e2e_out, sa, first_range);
            first_range = false;
            if (rc != PKDG_OK) break;
            if (cudaEventRecord(ctx->t_ev[1], sa) != cudaSuccess || cudaStreamWaitEvent(sb, ctx->t_ev[1], 0) != cudaSuccess) { rc = PKDG_ECUDA; break; }
            const int64_t r0 = Bh->first[b0], r1 = (int64_t)Bh->first[b1 - 1] + Bh->count[b1 - 1];
            if (r1 > r0 && cudaMemcpyAsync(out_host + 4 * r0, ctx->e2e_out + 4 * r0, sizeof(float) * 4 * (size_t)(r1 - r0),
                                           cudaMemcpyDeviceToHost, sb) != cudaSuccess) { rc = PKDG_ECUDA; break; }
        }
        return rc;
    };
    pkdg_status rc = run();
    cudaError_t e1 = cudaStreamSynchronize(sa), e2 = cudaStreamSynchronize(sb);   // also on the error path
    if (rc == PKDG_OK && (e1 != cudaSuccess || e2 != cudaSuccess)) rc = fail(ctx, PKDG_ECUDA, cudaGetErrorString(e1 != cudaSuccess ? e1 : e2));
    if (rc == PKDG_ECUDA && ctx->err.empty()) ctx->err = cudaGetErrorString(cudaGetLastError());
    ctx->last_stream = sa; ctx->last_chunks = n_ranges; ctx->last_buckets = nb;
    return rc;
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
    out->fixup_sinks = (int64_t)h.fixup_sinks;
    out->invalid_values = (int64_t)h.invalid_values;
    out->invalid_pairs = (int64_t)h.invalid_pairs;
    out->interactions_cc = (int64_t)h.interactions_cc;
    out->interactions_cp = (int64_t)h.interactions_cp;
    out->chunks = ctx->last_chunks;
    if (h.bad_entries) return fail(ctx, PKDG_EBADLIST, "validation found malformed buckets or list entries");
    if (h.invalid_values || h.invalid_pairs)
        return fail(ctx, PKDG_EBADVALUE, "PKDG_VALIDATE: values outside the documented range, or a sink inside a listed cell's b_max");
    return PKDG_OK;
}

pkdg_status pkdg_profile_enable(pkdg_ctx* ctx, int32_t on) {
    if (!ctx) return PKDG_EINVAL;
    ctx->profiling = on != 0;
    return PKDG_OK;
}

pkdg_status pkdg_profile_read(pkdg_ctx* ctx, int64_t* n, double* ms_total, double* fixup_ms_total) {
    if (!ctx || !n || !ms_total) return PKDG_EINVAL;
    CK(cudaSetDevice(ctx->device));
    double tot = 0, fix = 0;
    for (int i = 0; i < ctx->prof_n; ++i) {
        float ms = 0;
        CK(cudaEventSynchronize(ctx->prof_ev[3 * i + 2]));
        CK(cudaEventElapsedTime(&ms, ctx->prof_ev[3 * i], ctx->prof_ev[3 * i + 1]));
        tot += ms;
        CK(cudaEventElapsedTime(&ms, ctx->prof_ev[3 * i + 1], ctx->prof_ev[3 * i + 2]));
        fix += ms;
    }
    *n = ctx->prof_n;
    *ms_total = tot;
    if (fixup_ms_total) *fixup_ms_total = fix;
    ctx->prof_n = 0;
    return PKDG_OK;
}

pkdg_status pkdg_set_option(pkdg_ctx* ctx, int32_t option, double value) {
    if (!ctx) return PKDG_EINVAL;
    switch (option) {
        case PKDG_OPT_KAPPA2:
            if (!(value > 0.0) || value > 1.0e15) return fail(ctx, PKDG_EINVAL, "PKDG_OPT_KAPPA2 must be > 0");
            ctx->kappa2 = (float)value;
            return PKDG_OK;
        default: return fail(ctx, PKDG_EINVAL, "unknown option");
    }
}

int64_t pkdg_launch_count(const pkdg_ctx* ctx) { return ctx ? ctx->launches : 0; }

const char* pkdg_status_string(pkdg_status s) {
    switch (s) {
        case PKDG_OK: return "PKDG_OK";
        case PKDG_EINVAL: return "PKDG_EINVAL: invalid argument";
        case PKDG_ECUDA: return "PKDG_ECUDA: CUDA runtime error";
        case PKDG_ENOMEM: return "PKDG_ENOMEM: out of memory";
        case PKDG_EBADLIST: return "PKDG_EBADLIST: malformed buckets or lists";
        case PKDG_EBADVALUE: return "PKDG_EBADVALUE: values or geometry outside the documented range";
        default: return "unknown pkdg_status";
    }
}

const char* pkdg_last_error(const pkdg_ctx* ctx) { return ctx ? ctx->err.c_str() : g_create_err.c_str(); }

void pkdg_version(int32_t* major, int32_t* minor) {
    if (major) *major = PKDG_VERSION_MAJOR;
    if (minor) *minor = PKDG_VERSION_MINOR;
}

pkdg_status pkdg_fma_peak_probe(pkdg_ctx* ctx, int64_t iters, float* ms_host, double* flops_host) {
    if (!ctx || !ms_host || !flops_host || iters < 1) return PKDG_EINVAL;
    CK(cudaSetDevice(ctx->device));
    const int threads = 256, blocks = ctx->num_sms * 8;
    float* buf = nullptr;
    CK(cudaMalloc((void**)&buf, sizeof(float) * threads * blocks));
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0));
    CK(cudaEventCreate(&e1));
    pkdg_fma_probe_kernel<<<blocks, threads>>>(buf, 16, 0.999f, 0.001f);  // warm-up
    CK(cudaEventRecord(e0, 0));
    pkdg_fma_probe_kernel<<<blocks, threads>>>(buf, iters, 0.999f, 0.001f);
    CK(cudaEventRecord(e1, 0));
    CK(cudaEventSynchronize(e1));
    ctx->launches += 2;
    CK(cudaGetLastError());
    CK(cudaEventElapsedTime(ms_host, e0, e1));
    *flops_host = 2.0 * 64.0 * (double)iters * (double)threads * blocks;  // 64 FFMA per trip and thread
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    CK(cudaFree(buf));
    return PKDG_OK;
}

}  // extern "C"
