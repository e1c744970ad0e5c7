// pkdg_kernels.cuh -- device code of pkdg-b200 (sm_100a).  See include/pkdg.h for the
// problem statement and DESIGN.md for the kernel design and its roofline.
//
// Kernels:
//   pkdg_prep_cells_kernel   canonical raw-moment records -> normalised trace-free records (128 B)
//   pkdg_pack_kernel         a1: bucket work descriptors, tile counts, validation, I_pp / I_pc
//   pkdg_tiles_kernel        a1: materialised 32-entry tiles (pkdg_pack_export)
//   pkdg_evalb_kernel        a2-a5 for per-bucket lists (the headline kernel): one warp per bucket, a lane owns a
//                            sink pair (packed FP32x2 arithmetic), sources stream through shared memory (cp.async);
//                            per-sink conditioning estimate, ill-conditioned sinks are queued
//   pkdg_evalg_kernel        the same for lists shared by a group of <= 64 sinks: one warp per group
//   pkdg_fixup_kernel        queued sinks re-evaluated with fp64 terms and fp64 accumulators
//   pkdg_walk_kernel         list construction: the tree walk with the opening criterion, bit-identical to the host's
//   pkdg_validate_*_kernel   PKDG_VALIDATE
//   pkdg_fma_probe_kernel    FFMA-only probe (roofline denominator check)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <type_traits>

namespace pkdg {

constexpr int kCellQFloats = 32;   // internal record: one 128-byte line
constexpr float kFar = 1.0e15f;    // position of a masked (padding) source: contributes exactly 0

struct __align__(16) BucketDesc {
    int32_t first, count, pp_len, pc_len;
    int64_t pp_begin, pc_begin;  // entry offsets relative to the idx pointers given to the kernel
};

struct DevStats {
    unsigned long long interactions_pp, interactions_pc, tiles_pp, tiles_pc, bad_entries, fixup_sinks;
    unsigned long long invalid_values, invalid_pairs;  // PKDG_VALIDATE
    unsigned long long interactions_cc, interactions_cp;  // pkdg_gravity_eval_fmm: entries of the C-C / C-P lists
};

// ------------------------------------------------------------------------------------------------
// Cell preparation.  Raw moments M^(n) (n = 2,3,4) -> symmetric trace-free Q^(n) = STF[M^(n)], then
// q^(n) = n c_n Q^(n) / (M s^n) with c_n = (2n-1)!!/n! = 3/2, 5/2, 35/8 and s the cell's length scale
// (b_max).  With d = x - COM, r = |d| and the scaled displacement tau = s d / r^2 (|tau| = s/r < 1):
//   V_n = q^(n) . tau^(n-1)  (vector),   e_n = V_n . tau  (= n c_n Q^(n).d^n / (M r^2n))
//   phi = -(M/r) [1 + sum_n e_n / n]
//   a   =  (M/r^3) [s G - S d],   G = sum_n V_n,   S = 1 + sum_n (2n+1)/n e_n
// which is the truncated Taylor series of include/pkdg.h (d^n(1/r) is trace-free, so contracting the
// raw moments with it equals contracting their trace-free part with d^n; the polynomials are
// homogeneous, so evaluating them at tau absorbs every power of s/r).  Arithmetic in fp64: the
// trace removal cancels leading digits.
// Every slice q_i.. of a trace-free tensor is trace-free itself, so V_n,i = sum q_i jk.. tau_j tau_k .. needs no
// component with two z indices among jk..: q_i..zz = -q_i..xx - q_i..yy moves the z^2 into the monomials
// (pc_body2: 5 terms instead of 6 at order 3, 7 instead of 10 at order 4).  What is stored is therefore every
// component with at most ONE z among the indices after the first -- the 5 + 7 + 9 independent ones and the six
// the i = z slices need besides.  Layout of the 32 floats (one 128-byte line):
//   0-3 COM, M | 4 s | 5-10 q2 xx xy xz yy yz zz | 11-19 q3 xxx xxy xxz xyy xyz yyy yyz xzz yzz |
//   20-31 q4 xxxx xxxy xxxz xxyy xxyz xyyy xyyz yyyy yyyz xxzz xyzz yyzz
// ------------------------------------------------------------------------------------------------
// One thread per cell; the 36-float records of a block's 128 cells are staged through shared memory so
// that global reads and writes are coalesced (a thread reading its own 144-byte record directly runs at
// a fifth of the HBM rate).  Row strides 37 / 33 floats keep the per-thread accesses bank-conflict-free.
constexpr int kPrepThreads = 128;
__device__ __forceinline__ void prep_one_cell(const float* __restrict__ r, float* __restrict__ o);

__global__ void __launch_bounds__(kPrepThreads) pkdg_prep_cells_kernel(const float* __restrict__ rec, int64_t n,
                                                                       int stride, float* __restrict__ out) {
    __shared__ float s_in[kPrepThreads * 37];
    __shared__ float s_out[kPrepThreads * 33];
    const int64_t c0 = (int64_t)blockIdx.x * kPrepThreads;
    const int nc = (int)min((int64_t)kPrepThreads, n - c0);
    for (int i = threadIdx.x; i < nc * 36; i += kPrepThreads) {
        const int row = i / 36, col = i - row * 36;
        s_in[row * 37 + col] = rec[(c0 + row) * (int64_t)stride + col];
    }
    __syncthreads();
    if ((int)threadIdx.x < nc) prep_one_cell(s_in + threadIdx.x * 37, s_out + threadIdx.x * 33);
    __syncthreads();
    for (int i = threadIdx.x; i < nc * kCellQFloats; i += kPrepThreads) {
        const int row = i >> 5, col = i & 31;
        out[c0 * kCellQFloats + i] = s_out[row * 33 + col];
    }
}

// fp64 core: q[0..31] in the layout above (shared by the fp32 record writer and the fp64 fix-up kernel)
__device__ __forceinline__ void prep_cell_f64(const float* __restrict__ r, double* __restrict__ o) {
    double M = r[3];
    const float* m2 = r + 4;
    const float* m3 = r + 10;
    const float* m4 = r + 20;
    // order 2: xx xy xz yy yz zz
    double tr2 = (double)m2[0] + m2[3] + m2[5];
    double q2[6] = {m2[0] - tr2 / 3, m2[1], m2[2], m2[3] - tr2 / 3, m2[4], m2[5] - tr2 / 3};
    // order 3: xxx xxy xxz xyy xyz xzz yyy yyz yzz zzz
    double Tx = (double)m3[0] + m3[3] + m3[5], Ty = (double)m3[1] + m3[6] + m3[8], Tz = (double)m3[2] + m3[7] + m3[9];
    double q3[10] = {m3[0] - 0.6 * Tx, m3[1] - 0.2 * Ty, m3[2] - 0.2 * Tz, m3[3] - 0.2 * Tx, m3[4],
                     m3[5] - 0.2 * Tx, m3[6] - 0.6 * Ty, m3[7] - 0.2 * Tz, m3[8] - 0.2 * Ty, m3[9] - 0.6 * Tz};
    // order 4: xxxx xxxy xxxz xxyy xxyz xxzz xyyy xyyz xyzz xzzz yyyy yyyz yyzz yzzz zzzz
    double Txx = (double)m4[0] + m4[3] + m4[5], Txy = (double)m4[1] + m4[6] + m4[8], Txz = (double)m4[2] + m4[7] + m4[9];
    double Tyy = (double)m4[3] + m4[10] + m4[12], Tyz = (double)m4[4] + m4[11] + m4[13], Tzz = (double)m4[5] + m4[12] + m4[14];
    double TT = Txx + Tyy + Tzz;
    const double i7 = 1.0 / 7.0, i35 = 1.0 / 35.0;
    double q4[15] = {m4[0] - 6 * i7 * Txx + 3 * i35 * TT, m4[1] - 3 * i7 * Txy, m4[2] - 3 * i7 * Txz,
                     m4[3] - i7 * (Txx + Tyy) + i35 * TT, m4[4] - i7 * Tyz, m4[5] - i7 * (Txx + Tzz) + i35 * TT,
                     m4[6] - 3 * i7 * Txy, m4[7] - i7 * Txz, m4[8] - i7 * Txy, m4[9] - 3 * i7 * Txz,
                     m4[10] - 6 * i7 * Tyy + 3 * i35 * TT, m4[11] - 3 * i7 * Tyz, m4[12] - i7 * (Tyy + Tzz) + i35 * TT,
                     m4[13] - 3 * i7 * Tyz, m4[14] - 6 * i7 * Tzz + 3 * i35 * TT};
    double s = r[35];
    if (!(s > 0.0)) s = (M > 0.0 && tr2 > 0.0) ? sqrt(tr2 / M) : 0.0;
    double k2 = 0, k3 = 0, k4 = 0;
    if (s > 0.0 && M != 0.0) {
        k2 = 2 * 1.5 / (M * s * s);
        k3 = 3 * 2.5 / (M * s * s * s);
        k4 = 4 * 4.375 / (M * s * s * s * s);
    }
    o[0] = r[0]; o[1] = r[1]; o[2] = r[2]; o[3] = r[3];
    o[4] = s;
    o[5] = k2 * q2[0]; o[6] = k2 * q2[1]; o[7] = k2 * q2[2];        // xx xy xz
    o[8] = k2 * q2[3]; o[9] = k2 * q2[4]; o[10] = k2 * q2[5];       // yy yz zz
    o[11] = k3 * q3[0]; o[12] = k3 * q3[1]; o[13] = k3 * q3[2];     // xxx xxy xxz
    o[14] = k3 * q3[3]; o[15] = k3 * q3[4]; o[16] = k3 * q3[6];     // xyy xyz yyy
    o[17] = k3 * q3[7]; o[18] = k3 * q3[5]; o[19] = k3 * q3[8];     // yyz xzz yzz
    o[20] = k4 * q4[0]; o[21] = k4 * q4[1]; o[22] = k4 * q4[2];     // xxxx xxxy xxxz
    o[23] = k4 * q4[3]; o[24] = k4 * q4[4]; o[25] = k4 * q4[6];     // xxyy xxyz xyyy
    o[26] = k4 * q4[7]; o[27] = k4 * q4[10]; o[28] = k4 * q4[11];   // xyyz yyyy yyyz
    o[29] = k4 * q4[5]; o[30] = k4 * q4[8]; o[31] = k4 * q4[12];    // xxzz xyzz yyzz
}

__device__ __forceinline__ void prep_one_cell(const float* __restrict__ r, float* __restrict__ o) {
    double q[kCellQFloats];
    prep_cell_f64(r, q);
#pragma unroll
    for (int i = 0; i < kCellQFloats; ++i) o[i] = (float)q[i];
}

// ------------------------------------------------------------------------------------------------
// a1 packer.  One thread per bucket: work descriptor (sink range, list ranges relative to the idx
// pointers the evaluation kernel gets), tile counts, interaction counts, structural validation.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned long long warp_sum_u64(unsigned long long v) {
#pragma unroll
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// With leaf_idx != NULL (PKDG_PP_LEAVES) the P-P entries are references into gfc[n_g] = (first, count) of all
// buckets: I_pp counts the particles they stand for, tiles_pp two references per tile; a reference out of
// range or to a bucket of more than 16 particles is a bad entry.
__global__ void pkdg_pack_kernel(const int32_t* __restrict__ first, const int32_t* __restrict__ count,
                                 const int64_t* __restrict__ pp_off, const int64_t* __restrict__ pc_off,
                                 int64_t n_buckets, int64_t n_particles, int64_t pp_base, int64_t pc_base,
                                 BucketDesc* __restrict__ desc, DevStats* __restrict__ stats,
                                 unsigned int* __restrict__ work_counter, unsigned int* __restrict__ fix_count,
                                 const int32_t* __restrict__ leaf_idx,
                                 const int2* __restrict__ gfc, int64_t n_g) {
    int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long ipp = 0, ipc = 0, tpp = 0, tpc = 0, bad = 0;
    if (b == 0) { *work_counter = 0u; *fix_count = 0u; }
    if (b < n_buckets) {
        BucketDesc d;
        d.first = first[b];
        d.count = count[b];
        int64_t p0 = pp_off ? pp_off[b] : 0, p1 = pp_off ? pp_off[b + 1] : 0;
        int64_t c0 = pc_off ? pc_off[b] : 0, c1 = pc_off ? pc_off[b + 1] : 0;
        int64_t lp = p1 - p0, lc = c1 - c0;
        if (d.count < 0 || d.first < 0 || (int64_t)d.first + d.count > n_particles) { bad++; d.count = 0; }
        if (lp < 0 || lp > 0x7fffffffLL) { bad++; lp = 0; }
        if (lc < 0 || lc > 0x7fffffffLL) { bad++; lc = 0; }
        d.pp_len = (int32_t)lp; d.pc_len = (int32_t)lc;
        d.pp_begin = p0 - pp_base; d.pc_begin = c0 - pc_base;
        desc[b] = d;
        ipp = (unsigned long long)d.count * (unsigned long long)lp;
        ipc = (unsigned long long)d.count * (unsigned long long)lc;
        tpp = (unsigned long long)((lp + 31) >> 5);
        if (leaf_idx) {
            unsigned long long np = 0;
            for (int64_t e = 0; e < lp; ++e) {
                const int32_t g = leaf_idx[p0 - pp_base + e];
                if (g < 0) continue;  // padding
                if (g >= n_g) { bad++; continue; }
                const int2 fc = gfc[g];
                if (fc.y > 16 || fc.y < 0) { bad++; continue; }
                np += (unsigned long long)fc.y;
            }
            ipp = (unsigned long long)d.count * np;
            tpp = (unsigned long long)((lp + 1) >> 1);
        }
        tpc = (unsigned long long)((lc + 31) >> 5);
    }
    ipp = warp_sum_u64(ipp); ipc = warp_sum_u64(ipc); tpp = warp_sum_u64(tpp); tpc = warp_sum_u64(tpc);
    bad = warp_sum_u64(bad);
    if ((threadIdx.x & 31) == 0) {
        if (ipp) atomicAdd(&stats->interactions_pp, ipp);
        if (ipc) atomicAdd(&stats->interactions_pc, ipc);
        if (tpp) atomicAdd(&stats->tiles_pp, tpp);
        if (tpc) atomicAdd(&stats->tiles_pc, tpc);
        if (bad) atomicAdd(&stats->bad_entries, bad);
    }
}

// Group-shared lists (the walk stops at groups of up to 64 particles =
// 4 buckets and resolves the checklist into ONE P-P and ONE P-C list per group).  One thread per group: the
// work descriptor of every bucket of the group points at the group's lists.  Groups must tile the bucket range
// in order; a group that does not is a bad entry and gets no work (neither here nor in pkdg_evalg_kernel).
__global__ void pkdg_pack_groups_kernel(const int32_t* __restrict__ first, const int32_t* __restrict__ count,
                                        const int32_t* __restrict__ g_first, const int32_t* __restrict__ g_n,
                                        const int64_t* __restrict__ pp_off, const int64_t* __restrict__ pc_off,
                                        int64_t n_groups, int64_t n_buckets, int64_t n_particles, int64_t pp_base,
                                        int64_t pc_base, int64_t bucket_base, BucketDesc* __restrict__ desc,
                                        DevStats* __restrict__ stats, unsigned int* __restrict__ work_counter,
                                        unsigned int* __restrict__ fix_count, const int32_t* __restrict__ leaf_idx,
                                        const int2* __restrict__ gfc, int64_t n_g) {
    int64_t g = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long ipp = 0, ipc = 0, tpp = 0, tpc = 0, bad = 0;
    if (g == 0) { *work_counter = 0u; *fix_count = 0u; }
    if (g < n_groups) {
        int64_t b0 = (int64_t)g_first[g] - bucket_base, nb = g_n[g];
        const int64_t want = g == 0 ? 0 : (int64_t)g_first[g - 1] - bucket_base + g_n[g - 1];
        // a group that breaks the tiling gets no descriptors at all (its buckets keep the empty ones the caller's
        // memset left) and pkdg_evalg_kernel skips it under the same test: two overlapping groups must not race
        if (nb < 0 || b0 != want || b0 + nb > n_buckets || (g == n_groups - 1 && b0 + nb != n_buckets)) {
            bad++;
            nb = 0;
        }
        int64_t p0 = pp_off ? pp_off[g] : 0, p1 = pp_off ? pp_off[g + 1] : 0;
        int64_t c0 = pc_off ? pc_off[g] : 0, c1 = pc_off ? pc_off[g + 1] : 0;
        int64_t lp = p1 - p0, lc = c1 - c0;
        if (lp < 0 || lp > 0x7fffffffLL) { bad++; lp = 0; }
        if (lc < 0 || lc > 0x7fffffffLL) { bad++; lc = 0; }
        unsigned long long np = (unsigned long long)lp;
        unsigned long long tp = (unsigned long long)((lp + 31) >> 5);
        if (leaf_idx) {
            np = 0;
            for (int64_t e = 0; e < lp; ++e) {
                const int32_t r = leaf_idx[p0 - pp_base + e];
                if (r < 0) continue;  // padding
                if (r >= n_g) { bad++; continue; }
                const int2 fc = gfc[r];
                if (fc.y > 16 || fc.y < 0) { bad++; continue; }
                np += (unsigned long long)fc.y;
            }
            tp = (unsigned long long)((lp + 1) >> 1);
        }
        for (int64_t b = b0; b < b0 + nb; ++b) {
            BucketDesc d;
            d.first = first[b];
            d.count = count[b];
            if (d.count < 0 || d.first < 0 || (int64_t)d.first + d.count > n_particles) { bad++; d.count = 0; }
            d.pp_len = (int32_t)lp; d.pc_len = (int32_t)lc;
            d.pp_begin = p0 - pp_base; d.pc_begin = c0 - pc_base;
            desc[b] = d;
            ipp += (unsigned long long)d.count * np;
            ipc += (unsigned long long)d.count * (unsigned long long)lc;
            tpp += tp;
            tpc += (unsigned long long)((lc + 31) >> 5);
        }
    }
    ipp = warp_sum_u64(ipp); ipc = warp_sum_u64(ipc); tpp = warp_sum_u64(tpp); tpc = warp_sum_u64(tpc);
    bad = warp_sum_u64(bad);
    if ((threadIdx.x & 31) == 0) {
        if (ipp) atomicAdd(&stats->interactions_pp, ipp);
        if (ipc) atomicAdd(&stats->interactions_pc, ipc);
        if (tpp) atomicAdd(&stats->tiles_pp, tpp);
        if (tpc) atomicAdd(&stats->tiles_pc, tpc);
        if (bad) atomicAdd(&stats->bad_entries, bad);
    }
}

// (first, count) of every bucket as one 8-byte record: what a P-P leaf reference is resolved against.
__global__ void pkdg_fc_kernel(const int32_t* __restrict__ first, const int32_t* __restrict__ count, int64_t n,
                               int64_t n_particles, int2* __restrict__ out) {
    int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= n) return;
    int2 fc = make_int2(first[b], count[b]);
    if (fc.y < 0 || fc.x < 0 || (int64_t)fc.x + fc.y > n_particles) fc = make_int2(0, 0);
    out[b] = fc;
}

// The tile view of a list, shared by the evaluation kernel and pkdg_pack_export: entry `lane` of
// tile k of a list of `len` entries that starts at idx[begin].
__device__ __forceinline__ int32_t tile_entry(const int32_t* __restrict__ idx, int64_t begin, int32_t len,
                                              int32_t k, int lane) {
    int32_t e = k * 32 + lane;
    return e < len ? __ldg(idx + begin + e) : -1;
}

// tile_off[b] = number of tiles before bucket b (exclusive scan done by the host wrapper with a
// single-block scan kernel below); one warp per tile.
__global__ void pkdg_tile_count_kernel(const int64_t* __restrict__ off, int64_t n_buckets, int64_t* __restrict__ ntile) {
    int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (b < n_buckets) ntile[b] = (off[b + 1] - off[b] + 31) >> 5;
}

// In-place exclusive scan of n int64 values (+ total at [n]) by ONE block: debug / export path only.
__global__ void pkdg_scan_kernel(int64_t* __restrict__ v, int64_t n) {
    __shared__ int64_t s_part[1024];
    __shared__ int64_t s_carry;
    int tid = threadIdx.x, nt = blockDim.x;
    if (tid == 0) s_carry = 0;
    __syncthreads();
    for (int64_t base = 0; base < n; base += nt) {
        int64_t i = base + tid;
        int64_t x = i < n ? v[i] : 0;
        s_part[tid] = x;
        __syncthreads();
        for (int o = 1; o < nt; o <<= 1) {
            int64_t y = tid >= o ? s_part[tid - o] : 0;
            __syncthreads();
            s_part[tid] += y;
            __syncthreads();
        }
        int64_t incl = s_part[tid];
        int64_t carry = s_carry;
        if (i < n) v[i] = carry + incl - x;
        __syncthreads();
        if (tid == nt - 1) s_carry = carry + incl;
        __syncthreads();
    }
    if (tid == 0) v[n] = s_carry;
}

__global__ void pkdg_tiles_kernel(const int64_t* __restrict__ off, const int32_t* __restrict__ idx,
                                  int64_t n_buckets, const int64_t* __restrict__ tile_off,
                                  int32_t* __restrict__ tiles, int64_t capacity) {
    int lane = threadIdx.x & 31;
    int64_t warp = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    int64_t nwarps = ((int64_t)gridDim.x * blockDim.x) >> 5;
    for (int64_t b = warp; b < n_buckets; b += nwarps) {
        int64_t begin = off[b];
        int64_t len64 = off[b + 1] - begin;
        int32_t len = len64 < 0 ? 0 : (int32_t)len64;
        int64_t t0 = tile_off[b];
        int32_t nt = (len + 31) >> 5;
        for (int32_t k = 0; k < nt; ++k)
            if (t0 + k < capacity) tiles[(t0 + k) * 32 + lane] = tile_entry(idx, begin, len, k, lane);
    }
}

// ------------------------------------------------------------------------------------------------
// Evaluation kernels (a2-a5): shared parameters and pieces.  Sinks are processed in passes of up to 16 per bucket
// (pkdg_evalb_kernel) or 64 per group (pkdg_evalg_kernel); PAPER.md:L188 cuts lists at warp multiples and sends the
// remainder to the CPU -- here remainders are masked in place.
// ------------------------------------------------------------------------------------------------
constexpr int kTMax = 16;  // sinks per pass

struct EvalParams {
    const float4* xyzm;
    const float4* cellq;  // 8 float4 per cell
    const BucketDesc* desc;
    const int32_t* pp_idx;
    const int32_t* pc_idx;
    const int2* gfc;      // PKDG_PP_LEAVES: (first, count) of EVERY bucket a P-P entry may refer to
    int64_t n_gbuckets;
    float4* out;
    DevStats* stats;
    unsigned int* work_counter;
    int64_t n_buckets, n_particles, n_cells;
    float h2c;    // (2 eps)^2, the clamp of r^2 in the Newtonian fast path; at least 1e-24
    float eps;
    uint32_t flags;
    // conditioning estimate and fix-up queue
    const float* cells_raw;   // canonical records (fix-up kernel)
    int32_t cells_stride;
    float fix_k;              // a sink is queued iff S2 > fix_k |a|^2; < 0: never, 0: always
    int4* fix_queue;          // {bucket, t0 | wide << 31, lane ballot, 0}
    unsigned int* fix_count;
    unsigned int fix_cap;
    // group-shared lists (pkdg_evalg_kernel): group g = buckets g_first[g] - g_base .. + g_n[g] of `desc`
    const int32_t* g_first;
    const int32_t* g_n;
    int64_t n_groups;
    int64_t g_base;
};

// Cubic-spline pair factors (Monaghan-Lattanzio density of support h; u = r / h < 1): a -= m d g / h^3,
// phi += m w / h.  fp64: between u = 1/2 and 1 the polynomial cancels from terms of size 48 to a result of
// size 1, which fp32 cannot do to 1e-7.  Used by the rare softened-pair correction of the evaluation kernel
// and by the fix-up kernel.
__device__ __forceinline__ void spline_gw_f64(double u, double& g, double& w) {
    const double u2 = u * u;
    if (u < 0.5) {
        g = 32.0 / 3.0 + u2 * (-38.4 + 32.0 * u);
        w = -2.8 + u2 * (16.0 / 3.0 + u2 * (-9.6 + 6.4 * u));
    } else {
        const double iu = 1.0 / u;
        g = 64.0 / 3.0 + u * (-48.0 + u * (38.4 - (32.0 / 3.0) * u)) - iu * iu * iu / 15.0;
        w = -3.2 + iu / 15.0 + u2 * (32.0 / 3.0 + u * (-16.0 + u * (9.6 - (32.0 / 15.0) * u)));
    }
}

// Correction of one softened pair: what has to be ADDED to the clamped Newtonian pair the fast path booked
// (g_c = ri_c^3, w_c = -ri_c with ri_c = MUFU.RSQ(h^2)) to get the spline pair; d = x_sink - x_source.
__device__ __noinline__ float2 pp_soft_correction(float dx, float dy, float dz, float eps, float ric) {
    const double h = 2.0 * (double)eps, hi = 1.0 / h;
    const double r2 = (double)dx * dx + (double)dy * dy + (double)dz * dz;
    double g = 0.0, w = 0.0;   // eps == 0 and coincident: undefined, contributes nothing
    if (r2 < h * h) {
        spline_gw_f64(sqrt(r2) * hi, g, w);
        g *= hi * hi * hi;
        w *= hi;
    }
    const double rc = (double)ric;
    return make_float2((float)(g - rc * rc * rc), (float)(w + rc));
}

// MUFU.RSQ without the denormal pre-/post-scaling rsqrtf() emits (inputs here are never denormal).
__device__ __forceinline__ float rsqrt_approx(float x) {
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}


// A cell held in registers by one lane: the 32 floats of its record.
struct CellRegs {
    float cx, cy, cz, M, s;
    float xx, xy, xz, yy, yz, zz;
    float xxx, xxy, xxz, xyy, xyz, yyy, yyz, xzz, yzz;
    float xxxx, xxxy, xxxz, xxyy, xxyz, xyyy, xyyz, yyyy, yyyz, xxzz, xyzz, yyzz;
};

__device__ __forceinline__ void cell_unpack(CellRegs& c, const float4 f0, const float4 f1, const float4 f2,
                                            const float4 f3, const float4 f4, const float4 f5,
                                            const float4 f6, const float4 f7) {
    c.cx = f0.x; c.cy = f0.y; c.cz = f0.z; c.M = f0.w;
    c.s = f1.x; c.xx = f1.y; c.xy = f1.z; c.xz = f1.w;
    c.yy = f2.x; c.yz = f2.y; c.zz = f2.z; c.xxx = f2.w;
    c.xxy = f3.x; c.xxz = f3.y; c.xyy = f3.z; c.xyz = f3.w;
    c.yyy = f4.x; c.yyz = f4.y; c.xzz = f4.z; c.yzz = f4.w;
    c.xxxx = f5.x; c.xxxy = f5.y; c.xxxz = f5.z; c.xxyy = f5.w;
    c.xxyz = f6.x; c.xyyy = f6.y; c.xyyz = f6.z; c.yyyy = f6.w;
    c.yyyz = f7.x; c.xxzz = f7.y; c.xyzz = f7.z; c.yyzz = f7.w;
}


// ------------------------------------------------------------------------------------------------
// Asynchronous staging helpers (cp.async = LDGSTS): global -> shared memory without registers.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* q) { return (uint32_t)__cvta_generic_to_shared(q); }
__device__ __forceinline__ void cp_async16(void* dst, const void* src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(smem_u32(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait_pending() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

struct ListLens { int pp, pc; };
__device__ __forceinline__ ListLens eff_lens(const BucketDesc& d, bool do_pp, bool do_pc) {
    ListLens l;
    l.pp = (do_pp && d.count > 0) ? d.pp_len : 0;
    l.pc = (do_pc && d.count > 0) ? d.pc_len : 0;
    return l;
}

// ------------------------------------------------------------------------------------------------
// Packed FP32x2 arithmetic (sm_100 FFMA2 / FMUL2 / FADD2).
//
// Measured on B200 (round 1, profiles/r01_bench_ng256.md): the register file delivers one 32-bit operand per bank
// (even / odd register) per clock, so a scalar FFMA with three distinct register operands issues every 1.5 clocks
// (0.66 of the FMA peak).  A packed FFMA2 computes two FMAs in two clocks from 64-bit register pairs (one read of
// each bank per operand) and accepts a scalar register broadcast to both halves: coefficient (scalar) x monomial
// (pair) + accumulator (pair) needs <= 2 reads per bank whenever one operand is reused from the previous
// instruction -- full FMA rate with half the issue slots -- and three clocks otherwise.  So the two halves of every
// packed value are two SINKS (a sink pair) and everything that belongs to a source is a scalar.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ float2 sp(float a) { return make_float2(a, a); }
__device__ __forceinline__ float2 neg2(float2 a) { return make_float2(-a.x, -a.y); }
__device__ __forceinline__ float2 f2mul(float2 a, float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ float2 f2add(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 f2fma(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }

// 2 v by an integer add to the exponent field: runs on the ALU pipe, not on the FMA pipe the kernel is bound by.
// Exact for normal numbers; 0 (a padding cell's tau) becomes 1.2e-38, which the products that follow flush to nothing.
// |v| < 1 here (tau = s d / r^2), so the exponent cannot overflow.
__device__ __forceinline__ float2 twice2(float2 v) {
    return make_float2(__int_as_float(__float_as_int(v.x) + 0x00800000), __int_as_float(__float_as_int(v.y) + 0x00800000));
}

struct PcPre2 { float2 dx, dy, dz, ri; };

__device__ __forceinline__ PcPre2 pc_pre2(const float4 txy, const float4 tz, const CellRegs& c, float& minr2) {
    PcPre2 q;
    q.dx = f2add(make_float2(txy.x, txy.y), sp(-c.cx));
    q.dy = f2add(make_float2(txy.z, txy.w), sp(-c.cy));
    q.dz = f2add(make_float2(tz.x, tz.y), sp(-c.cz));
    const float2 r2 = f2fma(q.dz, q.dz, f2fma(q.dy, q.dy, f2mul(q.dx, q.dx)));
    q.ri = make_float2(rsqrt_approx(r2.x), rsqrt_approx(r2.y));
    minr2 = fminf(minr2, fminf(r2.x, r2.y));   // conditioning bound (min/max run on the ALU pipe, not the FMA pipe)
    return q;
}

// One cell against one sink pair, packed.  ONE cumulative chain per component: W2 = V2, W3 = W2 + V3,
// W4 = W3 + V4 = G (the order-3 chain starts from the order-2 result, the order-4 chain from the order-3 one).
// With E2 = W2.tau = e2, E3 = W3.tau = e2 + e3, E4 = G.tau = e2 + e3 + e4:
//   1 + sum e_n / n        = 1 + E2/6 + E3/12 + E4/4      (potential series fs)
//   1 + sum (2n+1)/n e_n   = fs + 2 E4                     (radial factor S)
// which needs no chain-start multiplies and no V2 + V3 + V4 sums.  The z^2 of every monomial is folded into the
// x^2 and y^2 ones (the slices are trace-free, see the record layout): with A = xx - zz, B = yy - zz,
//   V3_i = q_ixx A + q_iyy B + q_ixy 2xy + q_ixz 2xz + q_iyz 2yz
//   V4_i = q_ixxx x(xx - 3zz) + q_ixxy 3yA + q_ixxz z(3xx - zz) + q_ixyy 3xB + q_ixyz 6xyz
//        + q_iyyy y(yy - 3zz) + q_iyyz z(3yy - zz)
// Per interaction: 5 FADD, 31 FMUL, 65 FFMA, 1 MUFU = 167 flops in 101 packed instructions per pair, plus two
// doublings done as integer adds on the ALU pipe (the textbook form with all 6 + 10 monomials: 187 flops in 113).
#define PKDG_T0(CX, CY, CZ, M) vx = f2mul(sp(CX), M); vy = f2mul(sp(CY), M); vz = f2mul(sp(CZ), M);
#define PKDG_T1(CX, CY, CZ, M) vx = f2fma(sp(CX), M, vx); vy = f2fma(sp(CY), M, vy); vz = f2fma(sp(CZ), M, vz);
__device__ __forceinline__ void pc_body2(const PcPre2 q, const CellRegs& c, float4& a0, float4& a1) {
    const float2 ri2 = f2mul(q.ri, q.ri);
    const float2 sr = f2mul(sp(c.s), ri2);
    const float2 x = f2mul(q.dx, sr), y = f2mul(q.dy, sr), z = f2mul(q.dz, sr);  // tau
    float2 vx, vy, vz;
    PKDG_T0(c.xx, c.xy, c.xz, x) PKDG_T1(c.xy, c.yy, c.yz, y) PKDG_T1(c.xz, c.yz, c.zz, z)
    float2 E2 = f2mul(vx, x); E2 = f2fma(vy, y, E2); E2 = f2fma(vz, z, E2);
    const float2 xx = f2mul(x, x), yy = f2mul(y, y), zz = f2mul(z, z);
    const float2 A = f2add(xx, neg2(zz)), B = f2add(yy, neg2(zz));
    const float2 x2 = twice2(x), y2 = twice2(y);
    const float2 C = f2mul(x2, y), D = f2mul(x2, z), E = f2mul(y2, z);
    PKDG_T1(c.xxx, c.xxy, c.xxz, A) PKDG_T1(c.xyy, c.yyy, c.yyz, B) PKDG_T1(c.xxy, c.xyy, c.xyz, C)
    PKDG_T1(c.xxz, c.xyz, c.xzz, D) PKDG_T1(c.xyz, c.yyz, c.yzz, E)
    float2 E3 = f2mul(vx, x); E3 = f2fma(vy, y, E3); E3 = f2fma(vz, z, E3);
    const float2 P1 = f2fma(sp(-3.0f), zz, xx), P2 = f2fma(sp(3.0f), xx, neg2(zz));
    const float2 P3 = f2fma(sp(-3.0f), zz, yy), P4 = f2fma(sp(3.0f), yy, neg2(zz));
    const float2 x3 = f2mul(sp(3.0f), x), y3 = f2mul(sp(3.0f), y);
    const float2 K1 = f2mul(x, P1), K2 = f2mul(y3, A), K3 = f2mul(z, P2), K4 = f2mul(x3, B), K5 = f2mul(x3, E);
    const float2 K6 = f2mul(y, P3), K7 = f2mul(z, P4);
    PKDG_T1(c.xxxx, c.xxxy, c.xxxz, K1) PKDG_T1(c.xxxy, c.xxyy, c.xxyz, K2) PKDG_T1(c.xxxz, c.xxyz, c.xxzz, K3)
    PKDG_T1(c.xxyy, c.xyyy, c.xyyz, K4) PKDG_T1(c.xxyz, c.xyyz, c.xyzz, K5) PKDG_T1(c.xyyy, c.yyyy, c.yyyz, K6)
    PKDG_T1(c.xyyz, c.yyyz, c.yyzz, K7)
    float2 E4 = f2mul(vx, x); E4 = f2fma(vy, y, E4); E4 = f2fma(vz, z, E4);
    const float2 fs = f2fma(sp(0.25f), E4, f2fma(sp(0.083333333333f), E3, f2fma(sp(0.16666666667f), E2, sp(1.0f))));
    const float2 S = f2fma(sp(2.0f), E4, fs);
    const float2 mr = f2mul(sp(c.M), q.ri);
    const float2 k3 = f2mul(mr, ri2);
    const float2 sk = f2mul(sp(c.s), k3), Sk = f2mul(S, k3);
    float2 ax = make_float2(a0.x, a0.y), ay = make_float2(a0.z, a0.w), az = make_float2(a1.x, a1.y),
           aw = make_float2(a1.z, a1.w);
    aw = f2fma(neg2(mr), fs, aw);
    ax = f2fma(sk, vx, f2fma(neg2(Sk), q.dx, ax));
    ay = f2fma(sk, vy, f2fma(neg2(Sk), q.dy, ay));
    az = f2fma(sk, vz, f2fma(neg2(Sk), q.dz, az));
    a0 = make_float4(ax.x, ax.y, ay.x, ay.y);
    a1 = make_float4(az.x, az.y, aw.x, aw.y);
}
#undef PKDG_T0
#undef PKDG_T1

// Queue one (bucket, pass) for the fp64 fix-up kernel (warp-uniform call).  Returns false if the queue is full
// (cannot happen with the capacity the host sizes it to for non-overlapping buckets): the caller then writes
// the fp32 result instead of dropping the rows.
__device__ __forceinline__ bool fix_push(const EvalParams& p, int bucket, int t0w, unsigned ballot, int lane) {
    unsigned k = 0;
    if (lane == 0) {
        k = atomicAdd(p.fix_count, 1u);
        if (k < p.fix_cap) p.fix_queue[k] = make_int4(bucket, t0w, (int)ballot, 0);
    }
    k = __shfl_sync(0xffffffffu, k, 0);
    return k < p.fix_cap;
}

// ------------------------------------------------------------------------------------------------
// Group kernel (ONE P-P and ONE P-C list per group of up to 64 particles
// = 4 buckets).  With a list shared by 64 sinks the mapping turns round: one warp per group, one lane per SINK
// PAIR (the two halves of every packed value are the lane's two sinks, as before), and the SOURCES are
// warp-uniform: tiles of 32 source particles / 32 cell records stream through shared memory (cp.async, double
// buffered, coalesced: 8 lanes per 128-byte record) and every lane reads them by broadcast.  Consequences:
//   - sinks and accumulators live in registers for the whole list: no per-lane partial sums in shared memory,
//     no cross-lane reduction, no per-tile staging of 35 coefficients per lane;
//   - a list need not be a multiple of 32: cells are visited one by one, nothing is padded;
//   - index gather, bounds checks and staging are paid once per 64 sinks instead of once per 16;
//   - the conditioning estimate is the exact per-sink S2_i = sum_j |a_ij|^2 (one packed FMA per source);
//   - a softened pair is corrected in place (the lane owns its sinks).
// Arithmetic per interaction is that of pp_fast2 / pc_body2.
// ------------------------------------------------------------------------------------------------
constexpr int kGSinks = 64;   // sinks per pass of a group (2 per lane)

struct __align__(16) WarpSmemG {
    float4 cell[2][32 * 8];   // P-C tile: 32 internal cell records, double buffered
    float4 src[2][32];        // P-P tile: 32 source particles (x, y, z, m); padding = far away with mass 0
    int32_t sidx[2][32];      // their particle indices (self test by index), -1 = padding
    int32_t cidx[2][32];      // cell indices of the P-C tile being staged
    int32_t sink[kGSinks];    // particle index of sink slot t of the pass, -1 = none
    int32_t sbkt[kGSinks];    // its bucket (index into desc) and slot in that bucket: names it in the fix-up queue
    int32_t sslot[kGSinks];
};

// Coordinate c (0, 1, 2) of the sinks iA, iB of a lane as one packed pair; an unused slot (index < 0) is a dummy
// sink at -1e15 that no source comes near.
__device__ __forceinline__ float2 sink_pair_coord(const float4* __restrict__ xyzm, int iA, int iB, int c) {
    const float* f = reinterpret_cast<const float*>(xyzm);
    return make_float2(iA >= 0 ? __ldg(f + 4 * (int64_t)iA + c) : -kFar, iB >= 0 ? __ldg(f + 4 * (int64_t)iB + c) : -kFar);
}

// One source against the lane's sink pair, Newtonian with r^2 clamped from below at h2c, plus the exact conditioning estimate.
template <bool SELF>
__device__ __forceinline__ void pp_pair_g(const float2 X, const float2 Y, const float2 Z, const float4 s, bool selfA,
                                          bool selfB, float h2c, float& minr2, float2& ax, float2& ay, float2& az,
                                          float2& aw, float2& s2) {
    const float2 dx = f2add(X, sp(-s.x)), dy = f2add(Y, sp(-s.y)), dz = f2add(Z, sp(-s.z));
    float2 r2 = f2fma(dz, dz, f2fma(dy, dy, f2mul(dx, dx)));
    const float2 ri = make_float2(rsqrt_approx(fmaxf(r2.x, h2c)), rsqrt_approx(fmaxf(r2.y, h2c)));
    float2 nm = sp(-s.w);
    if (SELF) {
        nm.x = selfA ? 0.0f : nm.x; nm.y = selfB ? 0.0f : nm.y;
        r2.x = selfA ? 3.0e38f : r2.x; r2.y = selfB ? 3.0e38f : r2.y;
    }
    minr2 = fminf(minr2, fminf(r2.x, r2.y));
    const float2 nmri = f2mul(nm, ri);
    const float2 t = f2mul(nmri, ri);   // -m / r^2 = -|a_ij|
    const float2 nmg = f2mul(t, ri);
    ax = f2fma(nmg, dx, ax);
    ay = f2fma(nmg, dy, ay);
    az = f2fma(nmg, dz, az);
    aw = f2add(aw, nmri);
    s2 = f2fma(t, t, s2);
}

// Softened-pair correction for one sink (scalar): replaces the clamped Newtonian pair booked by pp_pair_g.
__device__ __forceinline__ void pp_soft_fix_g(float x, float y, float z, const float4 s, const EvalParams& p, float& ax,
                                              float& ay, float& az, float& aw, float& s2) {
    const float dx = x - s.x, dy = y - s.y, dz = z - s.z;
    const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
    if (r2 < p.h2c) {
        const float ri = rsqrt_approx(p.h2c);
        const float2 dgw = pp_soft_correction(dx, dy, dz, p.eps, ri);
        const float mg = s.w * dgw.x;
        ax = fmaf(-mg, dx, ax); ay = fmaf(-mg, dy, ay); az = fmaf(-mg, dz, az);
        aw = fmaf(s.w, dgw.y, aw);
        const float tc = s.w * ri * ri;   // booked (m / h^2)^2; a softened pair pulls with up to 2.6 m / h^2
        s2 = fmaf(15.0f * tc, tc, s2);
    }
}

// One cell against the lane's sink pair, accumulators in registers (pc_pre2 + pc_body2 + conditioning).
__device__ __forceinline__ void pc_pair_g(const float2 X, const float2 Y, const float2 Z, const CellRegs& c, float2& ax,
                                          float2& ay, float2& az, float2& aw, float2& s2) {
    float dummy = 3.0e38f;
    const PcPre2 q = pc_pre2(make_float4(X.x, X.y, Y.x, Y.y), make_float4(Z.x, Z.y, 0.f, 0.f), c, dummy);
    float4 a0 = make_float4(ax.x, ax.y, ay.x, ay.y), a1 = make_float4(az.x, az.y, aw.x, aw.y);
    pc_body2(q, c, a0, a1);
    ax = make_float2(a0.x, a0.y); ay = make_float2(a0.z, a0.w); az = make_float2(a1.x, a1.y); aw = make_float2(a1.z, a1.w);
    const float2 t = f2mul(f2mul(sp(c.M), q.ri), q.ri);   // M / r^2: the size of this cell's contribution
    s2 = f2fma(t, t, s2);
}

template <int WARPS, int MINB, bool LEAF>
__global__ void __launch_bounds__(WARPS * 32, MINB) pkdg_evalg_kernel(const EvalParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31;
    WarpSmemG& S = reinterpret_cast<WarpSmemG*>(smem_raw)[threadIdx.x >> 5];
    const float4 far4 = make_float4(kFar, kFar, kFar, 0.0f);
    const bool do_pp = !(p.flags & 0x2u), do_pc = !(p.flags & 0x4u), accumulate = (p.flags & 0x1u) != 0;
    const bool fix_on = p.fix_k >= 0.0f;
    unsigned bad = 0;

    for (;;) {
        unsigned gu = 0;
        if (lane == 0) gu = atomicAdd(p.work_counter, 1u);
        gu = __shfl_sync(0xffffffffu, gu, 0);
        if ((int64_t)gu >= p.n_groups) break;
        const int64_t gb0 = (int64_t)__ldg(p.g_first + gu) - p.g_base;
        const int gn = __ldg(p.g_n + gu);
        if (gn <= 0 || gb0 < 0 || gb0 + gn > p.n_buckets) continue;   // counted as a bad entry by the packer
        {   // the packer's tiling test: a group that does not start where the previous one ends (or, being the last one,
            // does not end where the buckets do) has no descriptors and is skipped
            const int64_t want = gu == 0 ? 0 : (int64_t)__ldg(p.g_first + gu - 1) - p.g_base + __ldg(p.g_n + gu - 1);
            if (gb0 != want || ((int64_t)gu == p.n_groups - 1 && gb0 + gn != p.n_buckets)) continue;
        }
        const BucketDesc d0 = p.desc[gb0];                              // every bucket of the group names the group's lists
        const int pp_len = do_pp ? d0.pp_len : 0, pc_len = do_pc ? d0.pc_len : 0;
        int nt = 0;
        for (int b = 0; b < gn; ++b) nt += p.desc[gb0 + b].count;

        for (int pass0 = 0; pass0 < nt; pass0 += kGSinks) {
            // ---- a2: the pass's sinks -> registers (lane l owns sink slots 2l and 2l + 1)
            __syncwarp();
            S.sink[lane] = -1; S.sink[lane + 32] = -1;
            __syncwarp();
            int off = 0, lo = 0x7fffffff, hi = -1;   // [lo, hi): particle index range of the pass's sinks (self test per tile)
            for (int b = 0; b < gn; ++b) {
                const BucketDesc db = p.desc[gb0 + b];
                for (int t = lane; t < db.count; t += 32) {
                    const int pos = off + t - pass0;
                    if (pos >= 0 && pos < kGSinks) {
                        S.sink[pos] = db.first + t; S.sbkt[pos] = (int32_t)(gb0 + b); S.sslot[pos] = t;
                    }
                }
                const int t_lo = max(0, pass0 - off), t_hi = min(db.count, pass0 + kGSinks - off);
                if (t_hi > t_lo) { lo = min(lo, db.first + t_lo); hi = max(hi, db.first + t_hi); }
                off += db.count;
            }
            __syncwarp();
            const int iA = S.sink[2 * lane], iB = S.sink[2 * lane + 1];
            const float4 dummy_tgt = make_float4(-kFar, -kFar, -kFar, 0.0f);
            const float2 X = sink_pair_coord(p.xyzm, iA, iB, 0), Y = sink_pair_coord(p.xyzm, iA, iB, 1), Z = sink_pair_coord(p.xyzm, iA, iB, 2);
            float2 ax = make_float2(0.f, 0.f), ay = ax, az = ax, aw = ax, s2 = ax;

            // ---- a3: P-P.  Tile k (32 sources) is computed from buffer k & 1 while tile k + 1 lands in the other.
            {
                const int ntile = LEAF ? (pp_len + 1) >> 1 : (pp_len + 31) >> 5;
                const int half = lane >> 4, slot = lane & 15;
                auto ref_of = [&](int k) -> int32_t {           // LEAF: bucket reference of this half-warp in tile k
                    const int r = 2 * k + half;
                    return r < pp_len ? __ldg(p.pp_idx + d0.pp_begin + r) : -1;
                };
                auto fc_of = [&](int32_t g) -> int2 {
                    if ((uint32_t)g >= (uint64_t)p.n_gbuckets) return make_int2(0, 0);   // counted as a bad entry by the packer
                    const int2 fc = __ldg(p.gfc + g);
                    return fc.y > 16 ? make_int2(0, 0) : fc;      // counted as a bad entry by the packer
                };
                auto idx_of = [&](int k) -> int32_t { return tile_entry(p.pp_idx, d0.pp_begin, pp_len, k, lane); };
                auto issue = [&](int32_t j, int buf) {           // the lane's source of a tile starts its way to shared memory
                    if ((uint32_t)j >= (uint64_t)p.n_particles) { bad += (j >= 0); j = -1; }
                    S.sidx[buf][lane] = j;
                    if (j >= 0) cp_async16(&S.src[buf][lane], p.xyzm + j);
                    else S.src[buf][lane] = far4;
                    cp_async_commit();
                };
                int32_t jn = -1, gnn = -1;   // non-LEAF: index of the tile after next;  LEAF: reference of the tile after next
                int2 fcn = make_int2(0, 0);  // LEAF: (first, count) of the next tile's reference
                if (LEAF) {
                    if (ntile > 0) { const int2 fc = fc_of(ref_of(0)); issue(slot < fc.y ? fc.x + slot : -1, 0); }
                    fcn = ntile > 1 ? fc_of(ref_of(1)) : make_int2(0, 0);
                    gnn = ntile > 2 ? ref_of(2) : -1;
                } else {
                    if (ntile > 0) issue(idx_of(0), 0);
                    jn = ntile > 1 ? idx_of(1) : -1;
                }
                for (int k = 0; k < ntile; ++k) {
                    const int buf = k & 1;
                    cp_async_wait_all();
                    __syncwarp();   // tile k is visible to the warp; everybody is done with the other buffer
                    if (k + 1 < ntile) {
                        if (LEAF) {
                            issue(slot < fcn.y ? fcn.x + slot : -1, buf ^ 1);
                            fcn = (k + 2 < ntile) ? fc_of(gnn) : make_int2(0, 0);
                            gnn = (k + 3 < ntile) ? ref_of(k + 3) : -1;
                        } else {
                            issue(jn, buf ^ 1);
                            jn = (k + 2 < ntile) ? idx_of(k + 2) : -1;
                        }
                    }
                    const int32_t jl = S.sidx[buf][lane];
                    const bool own = __any_sync(0xffffffffu, jl >= lo && jl < hi);   // tile may hold sinks of this pass
                    float minr2 = 3.0e38f;
                    if (own) {
#pragma unroll 4
                        for (int j = 0; j < 32; ++j) {
                            const int32_t sj = S.sidx[buf][j];
                            pp_pair_g<true>(X, Y, Z, S.src[buf][j], sj == iA, sj == iB, p.h2c, minr2, ax, ay, az, aw, s2);
                        }
                    } else {
#pragma unroll 8
                        for (int j = 0; j < 32; ++j)
                            pp_pair_g<false>(X, Y, Z, S.src[buf][j], false, false, p.h2c, minr2, ax, ay, az, aw, s2);
                    }
                    if (minr2 < p.h2c) {   // rare: a pair of this lane inside the softening (or coincident): the lane owns its sinks
                        for (int j = 0; j < 32; ++j) {
                            const float4 s = S.src[buf][j];
                            const int32_t sj = S.sidx[buf][j];
                            if (sj < 0) continue;
                            if (sj != iA) pp_soft_fix_g(X.x, Y.x, Z.x, s, p, ax.x, ay.x, az.x, aw.x, s2.x);
                            if (sj != iB) pp_soft_fix_g(X.y, Y.y, Z.y, s, p, ax.y, ay.y, az.y, aw.y, s2.y);
                        }
                    }
                }
            }

            // ---- a4: P-C.  Tile k = 32 cell records, copied by the whole warp (8 lanes per record) into buffer k & 1.
            {
                const int ntile = (pc_len + 31) >> 5;
                auto cidx_of = [&](int k) -> int32_t { return tile_entry(p.pc_idx, d0.pc_begin, pc_len, k, lane); };
                auto issue = [&](int32_t c, int buf) {
                    if ((uint32_t)c >= (uint64_t)p.n_cells) { bad += (c >= 0); c = -1; }
                    S.cidx[buf][lane] = c;
                    __syncwarp();
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        const int e = i * 32 + lane, rec = e >> 3, part = e & 7;
                        const int32_t ci = S.cidx[buf][rec];
                        if (ci >= 0) cp_async16(&S.cell[buf][e], p.cellq + (int64_t)ci * 8 + part);
                        else S.cell[buf][e] = part == 0 ? far4 : make_float4(0.f, 0.f, 0.f, 0.f);
                    }
                    cp_async_commit();
                };
                __syncwarp();
                if (ntile > 0) issue(cidx_of(0), 0);
                int32_t cn = ntile > 1 ? cidx_of(1) : -1;
                for (int k = 0; k < ntile; ++k) {
                    const int buf = k & 1;
                    cp_async_wait_all();
                    __syncwarp();
                    if (k + 1 < ntile) {
                        issue(cn, buf ^ 1);
                        cn = (k + 2 < ntile) ? cidx_of(k + 2) : -1;
                    }
                    const int ncell = min(32, pc_len - 32 * k);
                    const float4* rec = S.cell[buf];
#pragma unroll 2
                    for (int c = 0; c < ncell; ++c) {
                        CellRegs cr;
                        cell_unpack(cr, rec[8 * c], rec[8 * c + 1], rec[8 * c + 2], rec[8 * c + 3], rec[8 * c + 4],
                                    rec[8 * c + 5], rec[8 * c + 6], rec[8 * c + 7]);
                        pc_pair_g(X, Y, Z, cr, ax, ay, az, aw, s2);
                    }
                }
            }

            // ---- a5: no reduction -- the lane holds its sinks' totals.  Conditioning test, queue, write-back.
            {
                float4 rA = make_float4(ax.x, ay.x, az.x, aw.x), rB = make_float4(ax.y, ay.y, az.y, aw.y);
                if (accumulate) {   // the conditioning test is against the total the row will hold
                    if (iA >= 0) { const float4 o = p.out[iA]; rA.x += o.x; rA.y += o.y; rA.z += o.z; rA.w += o.w; }
                    if (iB >= 0) { const float4 o = p.out[iB]; rB.x += o.x; rB.y += o.y; rB.z += o.z; rB.w += o.w; }
                }
                const float a2A = fmaf(rA.z, rA.z, fmaf(rA.y, rA.y, rA.x * rA.x)), a2B = fmaf(rB.z, rB.z, fmaf(rB.y, rB.y, rB.x * rB.x));
                const bool fix_all = p.fix_k == 0.0f;   // PKDG_FIXUP_ALL; otherwise a strict test: a sink with nothing to sum (S2 = |a| = 0) is not ill-conditioned
                bool flagA = fix_on && iA >= 0 && (fix_all || s2.x > p.fix_k * a2A), flagB = fix_on && iB >= 0 && (fix_all || s2.y > p.fix_k * a2B);
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const bool flag = h ? flagB : flagA;
                    if (flag) {   // one queue entry per flagged sink, in the evaluation kernel's format (wide pass: lane 2 t)
                        const int t = S.sslot[2 * lane + h];
                        const unsigned k = atomicAdd(p.fix_count, 1u);
                        if (k < p.fix_cap)
                            p.fix_queue[k] = make_int4(S.sbkt[2 * lane + h], (int)((unsigned)(t & ~15) | 0x80000000u),
                                                       (int)(1u << (2 * (t & 15))), 0);
                        else if (h) flagB = false; else flagA = false;   // queue full (cannot happen): keep the fp32 row
                    }
                }
                if (iA >= 0 && !flagA) p.out[iA] = rA;
                if (iB >= 0 && !flagB) p.out[iB] = rB;
            }
        }
    }
    if (bad) atomicAdd(&p.stats->bad_entries, (unsigned long long)bad);
}

// ------------------------------------------------------------------------------------------------
// Bucket kernel (a2-a5 for per-bucket lists): one bucket per warp, buckets handed out in tree order through an
// atomic counter (neighbouring buckets share most of their sources, so these come from L2 / L1).  A lane OWNS a
// sink pair -- the two halves of every packed value are its two sinks -- and keeps sinks and accumulators in
// registers; the sources stream through shared memory.  A pass of ntp <= 16 sinks has npp = ceil(ntp / 2) sink
// pairs and the 32 lanes are laid out as npp pairs x ns = floor(32 / npp) source slots:
//     13 - 16 sinks: 8 pairs x 4 slots;  11, 12: 6 x 5;  9, 10: 5 x 6;  7, 8: 4 x 8;  5, 6: 3 x 10;  3, 4: 2 x 16;  1, 2: 1 x 32
// (30 of 32 lanes busy for 5 and 6 pairs, where a fixed 8-pair layout would leave 3 or 2 lanes of every 8 idle; a
// binary tree over clustered particles fills its buckets to anything between 8 and 16).  A tile of T = ns *
// floor(32 / ns) sources (32 or 30: a multiple of ns, so that every trip over a tile keeps all busy lanes busy) is
// staged by the whole warp (cp.async, one source particle / one 128-byte cell record per lane) and lane (slot,
// pair) evaluates sources slot, slot + ns, ... of the tile against its pair.
//   - a list is padded to a multiple of ns, not of 32: P-C lists fill 99 % of their slots;
//   - no accumulator traffic through shared memory; the cross-lane reduction at the end of a pass is a few shuffle
//     rounds of 10 values;
//   - the conditioning estimate is the exact per-sink S2_i = sum_j |a_ij|^2, a softened pair is corrected in place;
//   - 96 registers, 20 warps per SM: the load chain at the start of a bucket (counter, descriptor, sinks, indices,
//     sources) is hidden by the other warps, there is no hand-built hand-over between buckets.
// P-P source tiles sit in a ring of 4 (three tiles in flight: a tile is only ~130 instructions per lane), P-C tiles
// are double buffered and tile 0 is issued before the P-P phase.
// ------------------------------------------------------------------------------------------------

constexpr int kBRing = 4;         // P-P source tiles in shared memory: one in use, kBRing - 1 in flight
struct __align__(16) WarpSmemB {
    float4 cell[2][8 * 32];       // [float4 of the record][cell of the tile]: writes by lane = cell and reads by
                                  // slot = cell mod ns are both conflict-free
    float4 src[kBRing][32];
    int32_t sidx[kBRing][32];
};

// floor(x / d) for 0 <= x <= 32, 1 <= d <= 8 without an integer division (the quotient's fractional part is a
// multiple of 1 / d >= 1 / 8, so the reciprocal's rounding cannot move it across an integer)
__device__ __forceinline__ int small_div(int x, int d) {
    return __float2int_rd(fmaf((float)x, __frcp_rn((float)d), 0.01f));
}

// One pass (<= 16 sinks) of one bucket.
template <bool LEAF>
__device__ __forceinline__ void bucket_pass(const EvalParams& p, WarpSmemB& S, const BucketDesc& d, const int bucket,
                                            const int t0, const int ntp, const int pp_len, const int pc_len,
                                            const int lane, unsigned& bad) {
    const int npp = ntp > 12 ? 8 : (ntp + 1) >> 1;   // sink pairs of the layout
    const int ns = small_div(32, npp);                // source slots
    const int slot = small_div(lane, npp), pair = lane - slot * npp;
    const bool busy = slot < ns;
    const int lslot = busy ? slot : 0;                // idle lanes shadow slot 0 (their sinks are dummies, nothing is written)
    const int T = (ns & (ns - 1)) ? 30 : 32;          // sources / cells per tile: ns * floor(32 / ns) (ns = 5, 6, 10: 30)
    const float4 far4 = make_float4(kFar, kFar, kFar, 0.0f);
    const bool accumulate = (p.flags & 0x1u) != 0, fix_on = p.fix_k >= 0.0f;
    const int lo = d.first + t0, hi = lo + ntp;   // particle index range of the pass's sinks (self test per tile)
    const int iA = busy && 2 * pair < ntp ? lo + 2 * pair : -1, iB = busy && 2 * pair + 1 < ntp ? lo + 2 * pair + 1 : -1;
    const float4 dummy_tgt = make_float4(-kFar, -kFar, -kFar, 0.0f);
    // scalar loads: a float4 load would tie (x_A, x_B) to two different register quads and ptxas would re-pack the
    // pair with two MOVs in front of every packed instruction that reads it (4.5 MOVs per P-P visit)
    const float2 X = sink_pair_coord(p.xyzm, iA, iB, 0), Y = sink_pair_coord(p.xyzm, iA, iB, 1), Z = sink_pair_coord(p.xyzm, iA, iB, 2);
    float2 ax = make_float2(0.f, 0.f), ay = ax, az = ax, aw = ax, s2 = ax;

    // ---- the lane's cell of P-C tile 0 starts its way to shared memory under the P-P phase
    const int pc_ntile = T == 32 ? (pc_len + 31) >> 5 : (pc_len + 29) / 30;
    const int32_t* __restrict__ pc_list = p.pc_idx + d.pc_begin;   // n_particles, n_cells < 2^31 (checked by the host): 32-bit tests
    const uint32_t np32 = (uint32_t)p.n_particles, nc32 = (uint32_t)p.n_cells;
    auto cidx_of = [&](int k) -> int32_t { const int e = k * T + lane; return (lane < T && e < pc_len) ? __ldg(pc_list + e) : -1; };
    auto issue_cell = [&](int32_t c, int buf) {
        if ((uint32_t)c >= nc32) { bad += (c >= 0); c = -1; }
        float4* dst = &S.cell[buf][lane];
        if (c >= 0) {
            const float4* q = p.cellq + (int64_t)c * 8;
#pragma unroll
            for (int i = 0; i < 8; ++i) cp_async16(dst + 32 * i, q + i);
        } else {   // padding: a cell of mass 0 far away
            dst[0] = far4;
#pragma unroll
            for (int i = 1; i < 8; ++i) dst[32 * i] = make_float4(0.f, 0.f, 0.f, 0.f);
        }
        cp_async_commit();
    };
    __syncwarp();   // the previous pass / bucket is done with every buffer
    int32_t cn = -1;
    if (pc_ntile > 0) {
        issue_cell(cidx_of(0), 0);
        cn = pc_ntile > 1 ? cidx_of(1) : -1;
    }

    // ---- a3: P-P.  Tile k is computed from ring buffer k % kBRing while tiles k + 1 .. k + kBRing - 1 are in flight.
    //      LEAF (PKDG_PP_LEAVES): a tile is TWO bucket references, lanes 0-15 stage the particles of the first and
    //      lanes 16-31 those of the second (a bucket holds at most 16), so a tile always has 32 slots.
    auto pp_phase = [&](auto full_tag) {   // two copies of the P-P loop: full buckets (8 x 4 lanes, everything a constant) and the rest
        constexpr bool FULL = decltype(full_tag)::value;
        const int nsl = FULL ? 4 : ns, Tl = FULL ? 32 : T, lsl = FULL ? (lane >> 3) : lslot;
        constexpr int PD = kBRing - 1;
        const int TP = LEAF ? 32 : Tl;
        const int ntile = LEAF ? (pp_len + 1) >> 1 : TP == 32 ? (pp_len + 31) >> 5 : (pp_len + 29) / 30;
        const int half = lane >> 4, hslot = lane & 15;
        auto ref_of = [&](int k) -> int32_t {           // LEAF: bucket reference of this half-warp in tile k
            const int r = 2 * k + half;
            return r < pp_len ? __ldg(p.pp_idx + d.pp_begin + r) : -1;
        };
        auto fc_of = [&](int32_t g) -> int2 {
            if ((uint32_t)g >= (uint64_t)p.n_gbuckets) return make_int2(0, 0);   // counted as a bad entry by the packer
            const int2 fc = __ldg(p.gfc + g);
            return fc.y > 16 ? make_int2(0, 0) : fc;
        };
        const int32_t* __restrict__ pp_list = p.pp_idx + d.pp_begin;
        auto idx_of = [&](int k) -> int32_t { const int e = k * TP + lane; return (lane < TP && e < pp_len) ? __ldg(pp_list + e) : -1; };
        auto issue = [&](int32_t j, int buf) {           // the lane's source of a tile starts its way to shared memory
            if ((uint32_t)j >= np32) { bad += (j >= 0); j = -1; }
            S.sidx[buf][lane] = j;
            if (j >= 0) cp_async16(&S.src[buf][lane], p.xyzm + j);
            else S.src[buf][lane] = far4;
            cp_async_commit();
        };
        int32_t jn = -1, gnn = -1;
        int2 fcn = make_int2(0, 0);
        // tiles 0 .. PD - 1 start now (one commit group per tile, empty if the list is shorter: the group count stays uniform)
        if (LEAF) {
            int32_t g0[PD + 2];
#pragma unroll
            for (int t = 0; t < PD + 2; ++t) g0[t] = t < ntile ? ref_of(t) : -1;
            int2 fc0[PD + 1];
#pragma unroll
            for (int t = 0; t < PD + 1; ++t) fc0[t] = t < ntile ? fc_of(g0[t]) : make_int2(0, 0);
#pragma unroll
            for (int t = 0; t < PD; ++t) {
                if (t < ntile) issue(hslot < fc0[t].y ? fc0[t].x + hslot : -1, t);
                else cp_async_commit();
            }
            fcn = fc0[PD]; gnn = g0[PD + 1];
        } else {
            int32_t j0[PD + 1];
#pragma unroll
            for (int t = 0; t < PD + 1; ++t) j0[t] = t < ntile ? idx_of(t) : -1;
#pragma unroll
            for (int t = 0; t < PD; ++t) {
                if (t < ntile) issue(j0[t], t);
                else cp_async_commit();
            }
            jn = j0[PD];
        }
        for (int k = 0; k < ntile; ++k) {
            const int buf = k & (kBRing - 1);
            cp_async_wait_pending<PD - 1>();
            __syncwarp();   // tile k is visible to the warp; everybody is done with tile k - 1, whose buffer tile k + PD takes
            if (k + PD < ntile) {
                if (LEAF) {
                    issue(hslot < fcn.y ? fcn.x + hslot : -1, (k + PD) & (kBRing - 1));
                    fcn = (k + PD + 1 < ntile) ? fc_of(gnn) : make_int2(0, 0);
                    gnn = (k + PD + 2 < ntile) ? ref_of(k + PD + 2) : -1;
                } else {
                    issue(jn, (k + PD) & (kBRing - 1));
                    jn = (k + PD + 1 < ntile) ? idx_of(k + PD + 1) : -1;
                }
            } else {
                cp_async_commit();
            }
            // sources of this tile the lane visits: slot, slot + ns, ...; a short last tile ends early
            const int nsrc = LEAF ? 32 : min(TP, pp_len - TP * k);
            const int32_t jl = S.sidx[buf][lane];
            const bool own = __any_sync(0xffffffffu, jl >= lo && jl < hi);   // tile holds sinks of this pass
            const float4* src = S.src[buf];
            const int32_t* sid = S.sidx[buf];
            // LEAF tiles have 32 slots whatever ns is: the last trip of a 30-slot layout runs past the tile for some lanes
            auto ld_src = [&](int pos) -> float4 { return (LEAF && pos >= 32) ? far4 : src[pos]; };
            auto ld_sid = [&](int pos) -> int32_t { return (LEAF && pos >= 32) ? -1 : sid[pos]; };
            float minr2 = 3.0e38f;
            if (FULL) {   // a full bucket: straight-line code over the 8 visits of a tile (a short last tile ends in padding
                          // slots, which contribute exactly 0: cheaper than a second, looping copy of the code)
                const float4* s8 = src + (lane >> 3);
                if (!own) {
#pragma unroll
                    for (int it = 0; it < 8; ++it)
                        pp_pair_g<false>(X, Y, Z, s8[4 * it], false, false, p.h2c, minr2, ax, ay, az, aw, s2);
                } else {
                    const int32_t* i8 = sid + (lane >> 3);
#pragma unroll
                    for (int it = 0; it < 8; ++it) {
                        const int32_t sj = i8[4 * it];
                        pp_pair_g<true>(X, Y, Z, s8[4 * it], sj == iA, sj == iB, p.h2c, minr2, ax, ay, az, aw, s2);
                    }
                }
            } else if (own) {                        // a tile with own particles: self test by index
                // (trip counts are warp-uniform: slots beyond the end of a short tile hold padding, which contributes 0)
#pragma unroll 2
                for (int base = 0; base < nsrc; base += nsl) {
                    const int32_t sj = ld_sid(base + lsl);
                    pp_pair_g<true>(X, Y, Z, ld_src(base + lsl), sj == iA, sj == iB, p.h2c, minr2, ax, ay, az, aw, s2);
                }
            } else {
#pragma unroll 3
                for (int base = 0; base < nsrc; base += nsl)
                    pp_pair_g<false>(X, Y, Z, ld_src(base + lsl), false, false, p.h2c, minr2, ax, ay, az, aw, s2);
            }
            if (minr2 < p.h2c) {   // rare: a pair of this lane inside the softening (or coincident): the lane owns its sinks
                for (int base = 0; base < nsrc; base += nsl) {
                    const float4 s = ld_src(base + lsl);
                    const int32_t sj = ld_sid(base + lsl);
                    if (sj < 0) continue;
                    if (sj != iA) pp_soft_fix_g(X.x, Y.x, Z.x, s, p, ax.x, ay.x, az.x, aw.x, s2.x);
                    if (sj != iB) pp_soft_fix_g(X.y, Y.y, Z.y, s, p, ax.y, ay.y, az.y, aw.y, s2.y);
                }
            }
        }
    
    };
    if (npp == 8) pp_phase(std::true_type{}); else pp_phase(std::false_type{});

    // ---- a4: P-C.  Tile k = T cell records, one per lane (8 x cp.async of 16 bytes), in buffer k & 1; tile 0 was
    //      issued before the P-P phase.
    {
        for (int k = 0; k < pc_ntile; ++k) {
            const int buf = k & 1;
            cp_async_wait_all();
            __syncwarp();
            if (k + 1 < pc_ntile) {
                issue_cell(cn, buf ^ 1);
                cn = (k + 2 < pc_ntile) ? cidx_of(k + 2) : -1;
            }
            const int ncell = min(T, pc_len - T * k);
            const float4* rec = S.cell[buf];
            // warp-uniform trips; a short tile ends in padding cells.  Full buckets (8 x 4 lanes: a full tile is 8 trips)
            // run two trips per iteration -- ptxas then keeps a few more operands in the reuse cache (config 3 -0.8 %);
            // the other layouts have 5 or 6 trips per tile and lose 4 % that way.
            if (npp == 8) {
                const float4* r = rec + (lane >> 3);
#pragma unroll 2
                for (int base = 0; base < ncell; base += 4) {
                    CellRegs cr;
                    cell_unpack(cr, r[base], r[base + 32], r[base + 64], r[base + 96], r[base + 128], r[base + 160],
                                r[base + 192], r[base + 224]);
                    pc_pair_g(X, Y, Z, cr, ax, ay, az, aw, s2);
                }
            } else {
#pragma unroll 1
                for (int base = 0; base < ncell; base += ns) {
                    const float4* r = rec + base + lslot;
                    CellRegs cr;
                    cell_unpack(cr, r[0], r[32], r[64], r[96], r[128], r[160], r[192], r[224]);
                    pc_pair_g(X, Y, Z, cr, ax, ay, az, aw, s2);
                }
            }
        }
    }

    // ---- a5: the source slots of every sink pair are summed by shuffles; lanes of slot 0 test and write
    if (npp == 8) {
#pragma unroll
        for (int o = 16; o >= 8; o >>= 1) {
            ax.x += __shfl_xor_sync(0xffffffffu, ax.x, o); ax.y += __shfl_xor_sync(0xffffffffu, ax.y, o);
            ay.x += __shfl_xor_sync(0xffffffffu, ay.x, o); ay.y += __shfl_xor_sync(0xffffffffu, ay.y, o);
            az.x += __shfl_xor_sync(0xffffffffu, az.x, o); az.y += __shfl_xor_sync(0xffffffffu, az.y, o);
            aw.x += __shfl_xor_sync(0xffffffffu, aw.x, o); aw.y += __shfl_xor_sync(0xffffffffu, aw.y, o);
            s2.x += __shfl_xor_sync(0xffffffffu, s2.x, o); s2.y += __shfl_xor_sync(0xffffffffu, s2.y, o);
        }
    } else {   // any number of slots: slot s < step takes slot s + step, step = 16, 8, .. 1
        for (int step = 16; step >= 1; step >>= 1) {
            if (step >= ns) continue;   // warp-uniform
            const int o = step * npp;
            const bool take = slot < step && slot + step < ns;   // then lane + o <= 31
            auto add = [&](float& v) { const float t = __shfl_down_sync(0xffffffffu, v, o & 31); v += take ? t : 0.0f; };
            add(ax.x); add(ax.y); add(ay.x); add(ay.y); add(az.x); add(az.y); add(aw.x); add(aw.y); add(s2.x); add(s2.y);
        }
    }
    float4 rA = make_float4(ax.x, ay.x, az.x, aw.x), rB = make_float4(ax.y, ay.y, az.y, aw.y);
    const bool wA = slot == 0 && iA >= 0, wB = slot == 0 && iB >= 0;
    if (accumulate) {   // the conditioning test is against the total the row will hold
        if (wA) { const float4 o = p.out[iA]; rA.x += o.x; rA.y += o.y; rA.z += o.z; rA.w += o.w; }
        if (wB) { const float4 o = p.out[iB]; rB.x += o.x; rB.y += o.y; rB.z += o.z; rB.w += o.w; }
    }
    const float a2A = fmaf(rA.z, rA.z, fmaf(rA.y, rA.y, rA.x * rA.x)), a2B = fmaf(rB.z, rB.z, fmaf(rB.y, rB.y, rB.x * rB.x));
    const bool fix_all = p.fix_k == 0.0f;   // PKDG_FIXUP_ALL; otherwise a strict test: a sink with nothing to sum (S2 = |a| = 0) is not ill-conditioned
    bool flagA = fix_on && wA && (fix_all || s2.x > p.fix_k * a2A), flagB = fix_on && wB && (fix_all || s2.y > p.fix_k * a2B);
    // one queue entry per (bucket, pass) in the fix-up kernel's format: sink t of the pass is bit 2 t
    const unsigned mask = __reduce_or_sync(0xffffffffu, ((unsigned)flagA << (4 * pair)) | ((unsigned)flagB << (4 * pair + 2)));
    if (mask) {
        const bool queued = fix_push(p, bucket, (int)((unsigned)t0 | 0x80000000u), mask, lane);
        flagA = flagA && queued; flagB = flagB && queued;   // queue full (cannot happen): keep the fp32 rows
    }
    if (wA && !flagA) p.out[iA] = rA;
    if (wB && !flagB) p.out[iB] = rB;
}

template <int WARPS, int MINB, bool LEAF>
__global__ void __launch_bounds__(WARPS * 32, MINB) pkdg_evalb_kernel(const EvalParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31;
    WarpSmemB& S = reinterpret_cast<WarpSmemB*>(smem_raw)[threadIdx.x >> 5];
    const bool do_pp = !(p.flags & 0x2u), do_pc = !(p.flags & 0x4u);
    unsigned bad = 0;
    for (;;) {
        unsigned bu = 0;
        if (lane == 0) bu = atomicAdd(p.work_counter, 1u);
        bu = __shfl_sync(0xffffffffu, bu, 0);
        if ((int64_t)bu >= p.n_buckets) break;
        const BucketDesc d = p.desc[bu];
        const int pp_len = do_pp ? d.pp_len : 0, pc_len = do_pc ? d.pc_len : 0;
        for (int t0 = 0; t0 < d.count; t0 += kTMax) {
            const int ntp = min(kTMax, d.count - t0);
            bucket_pass<LEAF>(p, S, d, (int)bu, t0, ntp, pp_len, pc_len, lane, bad);
        }
    }
    if (bad) atomicAdd(&p.stats->bad_entries, (unsigned long long)bad);
}

// ------------------------------------------------------------------------------------------------
// fp64 fix-up ("accumulated in double precision").  The
// evaluation kernel queues every (bucket, pass) that holds a sink whose sum a_i = sum_j a_ij cancels so
// far that fp32 TERMS cannot deliver the tolerance; here one warp takes one queue entry and evaluates its
// flagged sinks over the same lists with fp64 terms and fp64 accumulators (the FP64 pipe of the B200,
// idle otherwise), lanes striding the sources, and writes their rows.  The arithmetic is the same
// algebra as the fp32 path (spline pair; normalised trace-free series), from the CANONICAL records.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ double warp_sum_f64(double v) {
#pragma unroll
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

__device__ __forceinline__ void pp_pair_f64(const double xi, const double yi, const double zi, const float4 s,
                                            const double h, double (&a)[4]) {
    const double dx = xi - (double)s.x, dy = yi - (double)s.y, dz = zi - (double)s.z;
    const double r2 = dx * dx + dy * dy + dz * dz;
    const double m = (double)s.w;
    if (r2 >= h * h) {
        if (r2 < 1.0e-24) return;  // eps == 0 and (nearly) coincident: contributes nothing (include/pkdg.h)
        const double ir = rsqrt(r2);
        const double g = m * ir * ir * ir;
        a[0] -= g * dx; a[1] -= g * dy; a[2] -= g * dz; a[3] -= m * ir;
    } else {
        const double hi = 1.0 / h;
        double g, w;
        spline_gw_f64(sqrt(r2) * hi, g, w);
        g *= m * hi * hi * hi;
        a[0] -= g * dx; a[1] -= g * dy; a[2] -= g * dz; a[3] += m * w * hi;
    }
}

// One cell (canonical record) against one sink in fp64: formulas above pkdg_prep_cells_kernel, plain form.
__device__ __noinline__ void pc_pair_f64(const double xi, const double yi, const double zi, const float* __restrict__ rec,
                                         double (&a)[4]) {
    double q[kCellQFloats];
    prep_cell_f64(rec, q);
    const double dx = xi - q[0], dy = yi - q[1], dz = zi - q[2], M = q[3], sc = q[4];
    const double r2 = dx * dx + dy * dy + dz * dz;
    const double ri = rsqrt(r2), ri2 = ri * ri, sr = sc * ri2;
    const double x = dx * sr, y = dy * sr, z = dz * sr;
    const double qxx = q[5], qxy = q[6], qxz = q[7], qyy = q[8], qyz = q[9], qzz = q[10];
    const double v2x = qxx * x + qxy * y + qxz * z, v2y = qxy * x + qyy * y + qyz * z, v2z = qxz * x + qyz * y + qzz * z;
    const double e2 = v2x * x + v2y * y + v2z * z;
    const double xxx = q[11], xxy = q[12], xxz = q[13], xyy = q[14], xyz = q[15], yyy = q[16], yyz = q[17];
    const double xzz = q[18], yzz = q[19], zzz = -(xxz + yyz);
    const double mxx = x * x, myy = y * y, mzz = z * z, mxy = 2 * x * y, mxz = 2 * x * z, myz = 2 * y * z;
    const double v3x = xxx * mxx + xyy * myy + xzz * mzz + xxy * mxy + xxz * mxz + xyz * myz;
    const double v3y = xxy * mxx + yyy * myy + yzz * mzz + xyy * mxy + xyz * mxz + yyz * myz;
    const double v3z = xxz * mxx + yyz * myy + zzz * mzz + xyz * mxy + xzz * mxz + yzz * myz;
    const double e3 = v3x * x + v3y * y + v3z * z;
    const double xxxx = q[20], xxxy = q[21], xxxz = q[22], xxyy = q[23], xxyz = q[24], xyyy = q[25], xyyz = q[26];
    const double yyyy = q[27], yyyz = q[28], xxzz = q[29], xyzz = q[30], yyzz = q[31];
    const double xzzz = -(xxxz + xyyz), yzzz = -(xxyz + yyyz), zzzz = -(xxzz + yyzz);
    const double c0 = mxx * x, c1 = myy * y, c2 = mzz * z, c3 = 3 * mxx * y, c4 = 3 * mxx * z, c5 = 3 * myy * x;
    const double c6 = 3 * myy * z, c7 = 3 * mzz * x, c8 = 3 * mzz * y, c9 = 6 * x * y * z;
    const double v4x = xxxx * c0 + xxxy * c3 + xxxz * c4 + xxyy * c5 + xxyz * c9 + xxzz * c7 + xyyy * c1 + xyyz * c6 + xyzz * c8 + xzzz * c2;
    const double v4y = xxxy * c0 + xxyy * c3 + xxyz * c4 + xyyy * c5 + xyyz * c9 + xyzz * c7 + yyyy * c1 + yyyz * c6 + yyzz * c8 + yzzz * c2;
    const double v4z = xxxz * c0 + xxyz * c3 + xxzz * c4 + xyyz * c5 + xyzz * c9 + xzzz * c7 + yyyz * c1 + yyzz * c6 + yzzz * c8 + zzzz * c2;
    const double e4 = v4x * x + v4y * y + v4z * z;
    const double fs = 1.0 + e2 / 2.0 + e3 / 3.0 + e4 / 4.0;
    const double Sr = 1.0 + 2.5 * e2 + (7.0 / 3.0) * e3 + 2.25 * e4;
    const double mr = M * ri, k3 = mr * ri2;
    a[3] -= mr * fs;
    a[0] += k3 * (sc * (v2x + v3x + v4x) - Sr * dx);
    a[1] += k3 * (sc * (v2y + v3y + v4y) - Sr * dy);
    a[2] += k3 * (sc * (v2z + v3z + v4z) - Sr * dz);
}

// One CTA of kFixThreads threads per queue entry; its flagged sinks one after the other, all threads striding
// the lists of the bucket (a flagged sink is rare, its lists may be thousands of entries long).
constexpr int kFixThreads = 128;
__global__ void __launch_bounds__(kFixThreads) pkdg_fixup_kernel(const EvalParams p) {
    __shared__ double s_red[4][kFixThreads / 32];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const unsigned n = min(*p.fix_count, p.fix_cap);
    const bool do_pp = !(p.flags & 0x2u), do_pc = !(p.flags & 0x4u), accumulate = (p.flags & 0x1u) != 0;
    const bool pp_leaves = (p.flags & 0x8u) != 0;
    const double h = 2.0 * (double)p.eps;
    for (unsigned e = blockIdx.x; e < n; e += gridDim.x) {
        const int4 ent = p.fix_queue[e];
        const BucketDesc d = p.desc[ent.x];
        const bool wide = ((unsigned)ent.y & 0x80000000u) != 0;
        const int t0 = (int)((unsigned)ent.y & 0x7fffffffu);
        const ListLens L = eff_lens(d, do_pp, do_pc);
        unsigned lanes = (unsigned)ent.z;  // ballot of the flagged lanes of the evaluation kernel's reduction
        const unsigned keep = wide ? 0x55555555u : 0x11111111u;   // one lane per sink: 2 t (wide) or 4 t
        lanes &= keep;
        if (tid == 0) atomicAdd(&p.stats->fixup_sinks, (unsigned long long)__popc(lanes));
        while (lanes) {
            const int bit = __ffs(lanes) - 1;
            lanes &= lanes - 1;
            const int i = d.first + t0 + (wide ? bit >> 1 : bit >> 2);
            const float4 xi4 = __ldg(p.xyzm + i);
            const double xi = xi4.x, yi = xi4.y, zi = xi4.z;
            double a[4] = {0.0, 0.0, 0.0, 0.0};
            if (pp_leaves) {   // a reference stands for <= 16 particles: 8 references per sweep of the CTA
                const int sub = tid >> 4, slot = tid & 15;
                for (int r = sub; r < L.pp; r += kFixThreads / 16) {
                    const int32_t g = __ldg(p.pp_idx + d.pp_begin + r);
                    if ((uint32_t)g >= (uint64_t)p.n_gbuckets) continue;
                    const int2 fc = __ldg(p.gfc + g);
                    const int j = fc.x + slot;
                    if (slot < fc.y && j != i && (uint32_t)j < (uint64_t)p.n_particles)
                        pp_pair_f64(xi, yi, zi, __ldg(p.xyzm + j), h, a);
                }
            } else {
                for (int r = tid; r < L.pp; r += kFixThreads) {
                    const int32_t j = __ldg(p.pp_idx + d.pp_begin + r);
                    if (j != i && (uint32_t)j < (uint64_t)p.n_particles) pp_pair_f64(xi, yi, zi, __ldg(p.xyzm + j), h, a);
                }
            }
            for (int r = tid; r < L.pc; r += kFixThreads) {
                const int32_t c = __ldg(p.pc_idx + d.pc_begin + r);
                if ((uint32_t)c < (uint64_t)p.n_cells) pc_pair_f64(xi, yi, zi, p.cells_raw + (int64_t)c * p.cells_stride, a);
            }
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                a[k] = warp_sum_f64(a[k]);
                if (lane == 0) s_red[k][wid] = a[k];
            }
            __syncthreads();
            if (tid == 0) {
                double r[4];
#pragma unroll
                for (int k = 0; k < 4; ++k) r[k] = (s_red[k][0] + s_red[k][1]) + (s_red[k][2] + s_red[k][3]);
                if (accumulate) {
                    const float4 old = p.out[i];
                    r[0] += old.x; r[1] += old.y; r[2] += old.z; r[3] += old.w;
                }
                p.out[i] = make_float4((float)r[0], (float)r[1], (float)r[2], (float)r[3]);
            }
            __syncthreads();
        }
    }
}

// ------------------------------------------------------------------------------------------------
// List construction on the device (PAPER.md:L65 checklist walk, L69 opening radius
// RO = b_max / theta and the 2-softenings gap, Table 3 "Opening criteria").  One thread per sink cell (a
// bucket, or a group cell for group-shared lists) walks the tree in depth-first pre-order through the
// skip list `end` (cell k's subtree is [k, end[k])): for source cell k and sink B (reading A6)
//   P-C   iff  k != B, count[k] >= 2, |COM_B - COM_k| > b_max,B + b_max,k / theta, gap(bbox_B, bbox_k) >= 2 eps
//   else  a leaf joins the P-P list whole (its particle indices, or ONE bucket reference with leaf_rank != NULL)
//   else  the cell is opened (k + 1 is its first child).
// Neighbouring threads are neighbouring sinks and take nearly the same path.  The arithmetic is fp64 with
// explicit round-to-nearest operations and no fused multiply-add, so that every accept / open decision --
// hence every offset and every index -- equals the host generator's (gcc, x86-64 SSE2) bit for bit.
// FILL = false counts the entries of each list, FILL = true writes them at the given offsets.
// ------------------------------------------------------------------------------------------------
struct TreeView {
    const int32_t* first; const int32_t* count; const int32_t* end; const int32_t* isleaf;
    const float* bblo; const float* bbhi;   // [n_cells][3]
    const float* rec; int32_t stride;       // canonical cell records: COM at [0..2], b_max at [35]
    int64_t n_cells;
    const int32_t* leaf_rank;               // NULL, or [n_cells]: bucket index of a leaf cell (PKDG_PP_LEAVES output)
};

// What the walk needs of a cell, gathered once per call into one 64-byte record (one cache line per visited cell
// instead of six: the canonical record's COM and b_max sit in two different lines, the boxes in two arrays, count /
// end / isleaf / first in four more).  The values are copies, so every decision stays bit-identical.
struct __align__(16) WalkNode {     // first 32-byte sector: what every visit reads; second: the box (read only by cells that
    float cx, cy, cz;              // pass the distance test) and b_max (read for the sink cell).  Centre of mass;
    int32_t count;                 // particles of the cell; bit 31 set = a leaf
    double ro;                     // b_max / theta (fp64, IEEE division: the value the host walk computes at every visit)
    int32_t end, entry;            // end of the subtree; a leaf's P-P entry: its first particle, or its rank (leaf references)
    float lox, loy, loz, hix;      // bounding box
    float hiy, hiz, bmax, pad;
};

// A subtree end outside (k, n_cells] would stall the walk (k = end must advance) or send it out of the array: it is
// clamped into that range and counted as a bad entry, like every other malformed input of the library.
__global__ void pkdg_walk_nodes_kernel(const TreeView T, double theta, WalkNode* __restrict__ nodes,
                                       DevStats* __restrict__ stats) {
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= T.n_cells) return;
    const float* r = T.rec + k * (int64_t)T.stride;
    WalkNode w;
    w.cx = r[0]; w.cy = r[1]; w.cz = r[2]; w.bmax = r[35];
    w.ro = __ddiv_rn((double)r[35], theta);
    w.lox = T.bblo[3 * k]; w.loy = T.bblo[3 * k + 1]; w.loz = T.bblo[3 * k + 2];
    w.hix = T.bbhi[3 * k]; w.hiy = T.bbhi[3 * k + 1]; w.hiz = T.bbhi[3 * k + 2];
    const bool leaf = T.isleaf[k] != 0;
    w.count = (T.count[k] & 0x7fffffff) | (leaf ? (int32_t)0x80000000u : 0);
    const int64_t e = T.end[k];
    w.end = (int32_t)(e <= k ? k + 1 : e > T.n_cells ? T.n_cells : e);
    if ((int64_t)w.end != e && stats) atomicAdd(&stats->bad_entries, 1ull);
    w.entry = (leaf && T.leaf_rank) ? T.leaf_rank[k] : T.first[k];
    w.pad = 0.0f;
    nodes[k] = w;
}

// leaf_rank[cell of bucket b] = b: what a P-P entry for that leaf is with PKDG_PP_LEAVES (only leaves are ever read)
__global__ void pkdg_leaf_rank_kernel(const int32_t* __restrict__ bucket_cell, int64_t n_buckets, int32_t* __restrict__ leaf_rank) {
    const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (b < n_buckets) leaf_rank[bucket_cell[b]] = (int32_t)b;
}

template <bool FILL>
__global__ void pkdg_walk_kernel(const WalkNode* __restrict__ nodes, int64_t n_cells, bool leaf_refs,
                                 const int32_t* __restrict__ sink_cell, int64_t n_sinks, double theta,
                                 double eps, int64_t* __restrict__ pp_len, int64_t* __restrict__ pc_len,
                                 const int64_t* __restrict__ pp_off, const int64_t* __restrict__ pc_off,
                                 int32_t* __restrict__ pp_idx, int32_t* __restrict__ pc_idx,
                                 DevStats* __restrict__ stats) {
    const int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n_sinks) return;
    const int64_t cb = sink_cell[s];
    if (cb < 0 || cb >= n_cells) {   // not a cell of this tree: empty lists, one bad entry (counted by the count pass)
        if (!FILL) { pp_len[s] = 0; pc_len[s] = 0; if (stats) atomicAdd(&stats->bad_entries, 1ull); }
        return;
    }
    const float4* nq = reinterpret_cast<const float4*>(nodes);
    const float4 b0 = __ldg(nq + 4 * cb), b1 = __ldg(nq + 4 * cb + 2), b2 = __ldg(nq + 4 * cb + 3);
    const double bx = b0.x, by = b0.y, bz = b0.z, bmaxB = b2.z;
    const double lob0 = b1.x, lob1 = b1.y, lob2 = b1.z;
    const double hib0 = b1.w, hib1 = b2.x, hib2 = b2.y;
    const double gap_min2 = __dmul_rn(__dmul_rn(4.0, eps), eps);
    int64_t npp = 0, npc = 0;
    int64_t wpp = FILL ? pp_off[s] : 0, wpc = FILL ? pc_off[s] : 0;
    int64_t k = 0;
    while (k < n_cells) {
        const float4 q0 = __ldg(nq + 4 * k);                                    // COM, count | leaf bit
        const int4 q3 = __ldg(reinterpret_cast<const int4*>(nq + 4 * k + 1));   // ro (two words), end, entry
        const int32_t cw = __float_as_int(q0.w), cnt = cw & 0x7fffffff, end = q3.z;
        const bool leaf = cw < 0;
        const double ro = __hiloint2double(q3.y, q3.x);
        bool accept = false;
        if (k != cb && cnt >= 2) {
            const double dx = __dsub_rn(bx, (double)q0.x), dy = __dsub_rn(by, (double)q0.y), dz = __dsub_rn(bz, (double)q0.z);
            const double d = __dsqrt_rn(__dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz)));
            if (d > __dadd_rn(bmaxB, ro)) {
                const float4 q1 = __ldg(nq + 4 * k + 2), q2 = __ldg(nq + 4 * k + 3);
                const double lok0 = q1.x, lok1 = q1.y, lok2 = q1.z;
                const double hik0 = q1.w, hik1 = q2.x, hik2 = q2.y;
                double g0 = 0.0, g1 = 0.0, g2 = 0.0, t;
                t = __dsub_rn(lok0, hib0); if (t > g0) g0 = t;
                t = __dsub_rn(lob0, hik0); if (t > g0) g0 = t;
                t = __dsub_rn(lok1, hib1); if (t > g1) g1 = t;
                t = __dsub_rn(lob1, hik1); if (t > g1) g1 = t;
                t = __dsub_rn(lok2, hib2); if (t > g2) g2 = t;
                t = __dsub_rn(lob2, hik2); if (t > g2) g2 = t;
                const double gg = __dadd_rn(__dadd_rn(__dmul_rn(g0, g0), __dmul_rn(g1, g1)), __dmul_rn(g2, g2));
                accept = gg >= gap_min2;
            }
        }
        if (accept) {
            if (FILL) pc_idx[wpc++] = (int32_t)k;
            ++npc;
            k = end;
        } else if (leaf) {   // a leaf joins the P-P list whole
            if (leaf_refs) {
                if (FILL) pp_idx[wpp++] = q3.w;
                ++npp;
            } else {
                if (FILL) {
                    const int32_t f = q3.w;
                    for (int32_t j = 0; j < cnt; ++j) pp_idx[wpp++] = f + j;
                }
                npp += cnt;
            }
            k = end;
        } else {
            k = k + 1;
        }
    }
    if (!FILL) { pp_len[s] = npp; pc_len[s] = npc; }
}

// Exclusive scan of n int64 values in three launches (block scans, scan of the block totals, add): v[i] ->
// sum_{j<i} v[j], total at v[n].  kScanBlock * kScanItems values per block; the middle launch is one block.
constexpr int kScanBlock = 256, kScanItems = 8;
__global__ void __launch_bounds__(kScanBlock) pkdg_scan_blocks_kernel(int64_t* __restrict__ v, int64_t n,
                                                                       int64_t* __restrict__ block_tot) {
    __shared__ int64_t s_warp[kScanBlock / 32];
    const int64_t base = ((int64_t)blockIdx.x * kScanBlock + threadIdx.x) * kScanItems;
    int64_t x[kScanItems], run = 0;
#pragma unroll
    for (int i = 0; i < kScanItems; ++i) { x[i] = base + i < n ? v[base + i] : 0; run += x[i]; }
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    int64_t inc = run;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const int64_t y = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += y; }
    if (lane == 31) s_warp[wid] = inc;
    __syncthreads();
    int64_t wpre = 0;
    for (int w = 0; w < wid; ++w) wpre += s_warp[w];
    int64_t pre = wpre + inc - run;
#pragma unroll
    for (int i = 0; i < kScanItems; ++i) { if (base + i < n) v[base + i] = pre; pre += x[i]; }
    if (threadIdx.x == kScanBlock - 1) block_tot[blockIdx.x] = wpre + inc;
}

__global__ void pkdg_scan_add_kernel(int64_t* __restrict__ v, int64_t n, const int64_t* __restrict__ block_pre,
                                     int64_t n_blocks) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) v[i] += block_pre[i / (kScanBlock * kScanItems)];
    else if (i == n) v[n] = block_pre[n_blocks];
}

// ------------------------------------------------------------------------------------------------
// PKDG_VALIDATE: the value-range contract of include/pkdg.h checked on the device (optional; not on the
// timed path).  Values: every coordinate finite and |x| <= 1e12, every mass / moment finite.  Pairs: every
// listed (sink, cell) pair has the sink OUTSIDE the cell's b_max sphere (the expansion diverges inside).
// ------------------------------------------------------------------------------------------------
__global__ void pkdg_validate_values_kernel(const float4* __restrict__ xyzm, int64_t n_particles,
                                            const float* __restrict__ rec, int64_t n_cells, int stride,
                                            DevStats* __restrict__ stats) {
    unsigned long long bad = 0;
    const int64_t tid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x, nth = (int64_t)gridDim.x * blockDim.x;
    for (int64_t i = tid; i < n_particles; i += nth) {
        const float4 q = xyzm[i];
        const bool ok = fabsf(q.x) <= 1.0e12f && fabsf(q.y) <= 1.0e12f && fabsf(q.z) <= 1.0e12f && isfinite(q.w);
        bad += !ok;   // NaN coordinates fail the <= tests
    }
    for (int64_t c = tid; c < n_cells; c += nth) {
        const float* r = rec + c * (int64_t)stride;
        bool ok = fabsf(r[0]) <= 1.0e12f && fabsf(r[1]) <= 1.0e12f && fabsf(r[2]) <= 1.0e12f;
        for (int k = 3; k < 36; ++k) ok = ok && isfinite(r[k]);
        bad += !ok;
    }
    bad = warp_sum_u64(bad);
    if ((threadIdx.x & 31) == 0 && bad) atomicAdd(&stats->invalid_values, bad);
}

__global__ void pkdg_validate_pairs_kernel(const EvalParams p) {
    const int lane = threadIdx.x & 31;
    const int64_t gw = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5, nw = ((int64_t)gridDim.x * blockDim.x) >> 5;
    unsigned long long bad = 0;
    for (int64_t b = gw; b < p.n_buckets; b += nw) {
        const BucketDesc d = p.desc[b];
        for (int e = lane; e < d.pc_len; e += 32) {
            const int32_t c = __ldg(p.pc_idx + d.pc_begin + e);
            if ((uint32_t)c >= (uint64_t)p.n_cells) continue;   // counted as a bad entry by the evaluation kernel
            const float4 cm = __ldg(p.cellq + (int64_t)c * 8);
            const float sc = __ldg(reinterpret_cast<const float*>(p.cellq + (int64_t)c * 8 + 1));
            for (int t = 0; t < d.count; ++t) {
                const float4 x = __ldg(p.xyzm + d.first + t);
                const float dx = x.x - cm.x, dy = x.y - cm.y, dz = x.z - cm.z;
                bad += !(dx * dx + dy * dy + dz * dz > sc * sc);
            }
        }
    }
    bad = warp_sum_u64(bad);
    if (lane == 0 && bad) atomicAdd(&p.stats->invalid_pairs, bad);
}

// ------------------------------------------------------------------------------------------------
// FFMA-only probe (pkdg_fma_peak_probe): FFMA with two constant-bank operands (one register read per
// FMA), registers only -- what the FP32 pipe delivers; the roofline denominator cross-check of bench.py.
// ------------------------------------------------------------------------------------------------
__global__ void pkdg_fma_probe_kernel(float* out, int64_t iters, float a, float b) {
    float v0 = threadIdx.x, v1 = v0 + 1, v2 = v0 + 2, v3 = v0 + 3, v4 = v0 + 4, v5 = v0 + 5, v6 = v0 + 6, v7 = v0 + 7;
    for (int64_t i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            v0 = fmaf(v0, a, b); v1 = fmaf(v1, a, b); v2 = fmaf(v2, a, b); v3 = fmaf(v3, a, b);
            v4 = fmaf(v4, a, b); v5 = fmaf(v5, a, b); v6 = fmaf(v6, a, b); v7 = fmaf(v7, a, b);
        }
    }
    out[(int64_t)blockIdx.x * blockDim.x + threadIdx.x] = v0 + v1 + v2 + v3 + v4 + v5 + v6 + v7;
}


}  // namespace pkdg
