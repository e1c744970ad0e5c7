// pkdg_kernels.cuh -- device code of pkdg-b200 (sm_100a).  See include/pkdg.h for the
// problem statement and DESIGN.md for the kernel design and its roofline.
//
// Kernels:
//   pkdg_prep_cells_kernel  canonical raw-moment records -> normalised trace-free records (128 B)
//   pkdg_pack_kernel        a1: bucket work descriptors, tile counts, validation, I_pp / I_pc
//   pkdg_tiles_kernel       a1: materialised 32-entry tiles (pkdg_pack_export)
//   pkdg_eval_kernel<TB>    a2-a5: one warp per bucket, lanes stride the source lists, TB sinks
//                           register-blocked per pass, butterfly transpose-reduction, float4 store
//   pkdg_fma_probe_kernel   FFMA-only loop (roofline denominator check)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace pkdg {

constexpr int kCellQFloats = 32;   // internal record: one 128-byte line
constexpr float kFar = 1.0e15f;    // position of a masked (padding) source: contributes exactly 0

struct __align__(16) BucketDesc {
    int32_t first, count, pp_len, pc_len;
    int64_t pp_begin, pc_begin;  // entry offsets relative to the idx pointers given to the kernel
};

struct DevStats {
    unsigned long long interactions_pp, interactions_pc, tiles_pp, tiles_pc, bad_entries;
};

// ------------------------------------------------------------------------------------------------
// Cell preparation.  Raw moments M^(n) (n = 2,3,4) -> symmetric trace-free Q^(n) = STF[M^(n)], then
// q^(n) = c_n Q^(n) / (M s^n) with c_n = (2n-1)!!/n! = 3/2, 5/2, 35/8 and s the cell's length scale
// (b_max).  With u = r/|r|, t = s/|r|:
//   phi = -(M/|r|) [1 + sum_n t^n P_n(u)],           P_n = q^(n) . u^n
//   a   =  (M/|r|^2) [W - S u],  W = sum_n n t^n V_n, V_n = q^(n) . u^(n-1), S = 1 + sum_n (2n+1) t^n P_n
// which is the truncated Taylor series of include/pkdg.h (d^n(1/r) is trace-free, so contracting the
// raw moments with it equals contracting their trace-free part with r^n).  Arithmetic in fp64: the
// trace removal cancels leading digits.  Layout of the 32 floats:
//   0-3 COM, M | 4 s | 5-9 q2 xx xy xz yy yz | 10-16 q3 xxx xxy xxz xyy xyz yyy yyz |
//   17-25 q4 xxxx xxxy xxxz xxyy xxyz xyyy xyyz yyyy yyyz | 26 q2zz 27 q3xzz 28 q3yzz 29 q3zzz
//   30 q4xxzz 31 q4yyzz          (the other four dependent q4 components are rebuilt in registers)
// ------------------------------------------------------------------------------------------------
__global__ void pkdg_prep_cells_kernel(const float* __restrict__ rec, int64_t n, int stride,
                                       float* __restrict__ out) {
    int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= n) return;
    const float* r = rec + c * (int64_t)stride;
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
        k2 = 1.5 / (M * s * s);
        k3 = 2.5 / (M * s * s * s);
        k4 = 4.375 / (M * s * s * s * s);
    }
    float* o = out + c * kCellQFloats;
    o[0] = r[0]; o[1] = r[1]; o[2] = r[2]; o[3] = r[3];
    o[4] = (float)s;
    o[5] = (float)(k2 * q2[0]); o[6] = (float)(k2 * q2[1]); o[7] = (float)(k2 * q2[2]);
    o[8] = (float)(k2 * q2[3]); o[9] = (float)(k2 * q2[4]);
    o[10] = (float)(k3 * q3[0]); o[11] = (float)(k3 * q3[1]); o[12] = (float)(k3 * q3[2]);
    o[13] = (float)(k3 * q3[3]); o[14] = (float)(k3 * q3[4]); o[15] = (float)(k3 * q3[6]);
    o[16] = (float)(k3 * q3[7]);
    o[17] = (float)(k4 * q4[0]); o[18] = (float)(k4 * q4[1]); o[19] = (float)(k4 * q4[2]);
    o[20] = (float)(k4 * q4[3]); o[21] = (float)(k4 * q4[4]); o[22] = (float)(k4 * q4[6]);
    o[23] = (float)(k4 * q4[7]); o[24] = (float)(k4 * q4[10]); o[25] = (float)(k4 * q4[11]);
    o[26] = (float)(k2 * q2[5]);
    o[27] = (float)(k3 * q3[5]); o[28] = (float)(k3 * q3[8]); o[29] = (float)(k3 * q3[9]);
    o[30] = (float)(k4 * q4[5]); o[31] = (float)(k4 * q4[12]);
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

__global__ void pkdg_pack_kernel(const int32_t* __restrict__ first, const int32_t* __restrict__ count,
                                 const int64_t* __restrict__ pp_off, const int64_t* __restrict__ pc_off,
                                 int64_t n_buckets, int64_t n_particles, int64_t pp_base, int64_t pc_base,
                                 BucketDesc* __restrict__ desc, DevStats* __restrict__ stats,
                                 unsigned int* __restrict__ work_counter) {
    int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long ipp = 0, ipc = 0, tpp = 0, tpc = 0, bad = 0;
    if (b == 0) *work_counter = 0u;
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
// Evaluation kernel.
// ------------------------------------------------------------------------------------------------
struct EvalParams {
    const float4* xyzm;
    const float4* cellq;  // 8 float4 per cell
    const BucketDesc* desc;
    const int32_t* pp_idx;
    const int32_t* pc_idx;
    float4* out;
    DevStats* stats;
    unsigned int* work_counter;
    int64_t n_buckets, n_particles, n_cells;
    float h2min;  // max(h^2, FLT_MIN): pairs with r^2 < h2min leave the Newtonian fast path
    float hinv;   // 1/h, 0 if eps == 0
    uint32_t flags;
};

// One P-P interaction: sink (tx,ty,tz) with source s (x,y,z,m).  `self` = the source IS the sink.
// Newtonian fast path: 3 sub, 1 mul + 2 fma, rsqrt, 3 mul, 3 fma, 1 fma = 19 flops (rsqrt = 1).
__device__ __forceinline__ void pp_interact(const float4 t, const float4 s, bool self, float h2min,
                                            float hinv, float& ax, float& ay, float& az, float& ph) {
    float dx = t.x - s.x, dy = t.y - s.y, dz = t.z - s.z;
    float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
    float g, w;  // a -= m d g ; phi += m w
    if (r2 < h2min) {
        // softened (or coincident) pair: cubic-spline kernel of support h, u = r/h   (rare path)
        float r = sqrtf(r2);
        float u = r * hinv;
        float u2 = u * u;
        if (self || hinv == 0.0f) {
            g = 0.0f; w = 0.0f;  // own index: skipped.  eps == 0 and r == 0: undefined, skipped.
        } else if (u < 0.5f) {
            g = fmaf(u2, fmaf(32.0f, u, -38.4f), 10.666666667f);
            w = fmaf(u2, fmaf(u2, fmaf(6.4f, u, -9.6f), 5.3333333333f), -2.8f);
        } else {
            float iu = 1.0f / u;
            float iu3 = iu * iu * iu;
            g = fmaf(u, fmaf(u, fmaf(-10.666666667f, u, 38.4f), -48.0f), 21.333333333f) - 0.066666666667f * iu3;
            w = fmaf(u2, fmaf(u, fmaf(u, fmaf(-2.1333333333f, u, 9.6f), -16.0f), 10.666666667f), -3.2f) +
                0.066666666667f * iu;
        }
        g *= hinv * hinv * hinv;
        w *= hinv;
    } else {
        float ri = rsqrtf(r2);
        float ri2 = ri * ri;
        g = ri * ri2;
        w = -ri;
    }
    float mg = s.w * g;
    ax = fmaf(-mg, dx, ax);
    ay = fmaf(-mg, dy, ay);
    az = fmaf(-mg, dz, az);
    ph = fmaf(s.w, w, ph);
}

// A cell held in registers by one lane (35 values; COM/M/s + 6 + 10 + 15 normalised components).
struct CellRegs {
    float cx, cy, cz, M, s;
    float xx, xy, xz, yy, yz, zz;
    float xxx, xxy, xxz, xyy, xyz, xzz, yyy, yyz, yzz, zzz;
    float xxxx, xxxy, xxxz, xxyy, xxyz, xxzz, xyyy, xyyz, xyzz, xzzz, yyyy, yyyz, yyzz, yzzz, zzzz;
};

__device__ __forceinline__ void cell_unpack(CellRegs& c, const float4 f0, const float4 f1, const float4 f2,
                                            const float4 f3, const float4 f4, const float4 f5,
                                            const float4 f6, const float4 f7) {
    c.cx = f0.x; c.cy = f0.y; c.cz = f0.z; c.M = f0.w;
    c.s = f1.x; c.xx = f1.y; c.xy = f1.z; c.xz = f1.w;
    c.yy = f2.x; c.yz = f2.y; c.xxx = f2.z; c.xxy = f2.w;
    c.xxz = f3.x; c.xyy = f3.y; c.xyz = f3.z; c.yyy = f3.w;
    c.yyz = f4.x; c.xxxx = f4.y; c.xxxy = f4.z; c.xxxz = f4.w;
    c.xxyy = f5.x; c.xxyz = f5.y; c.xyyy = f5.z; c.xyyz = f5.w;
    c.yyyy = f6.x; c.yyyz = f6.y; c.zz = f6.z; c.xzz = f6.w;
    c.yzz = f7.x; c.zzz = f7.y; c.xxzz = f7.z; c.yyzz = f7.w;
    c.xyzz = -(c.xxxy + c.xyyy);
    c.xzzz = -(c.xxxz + c.xyyz);
    c.yzzz = -(c.xxyz + c.yyyz);
    c.zzzz = -(c.xxzz + c.yyzz);
}

// One P-C interaction (see the formulas above pkdg_prep_cells_kernel).  ~130 FP32-pipe
// instructions + 1 MUFU; audited flop count in DESIGN.md.
__device__ __forceinline__ void pc_interact(const float4 t, const CellRegs& c, float& ax, float& ay,
                                            float& az, float& ph) {
    float dx = t.x - c.cx, dy = t.y - c.cy, dz = t.z - c.cz;
    float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
    float ri = rsqrtf(r2);
    // one Newton step: MUFU.RSQ is good to ~2^-22.9, and the result enters as ri^2..ri^6
    float hy = 0.5f * r2 * ri;
    ri = ri * fmaf(-hy, ri, 1.5f);
    float x = dx * ri, y = dy * ri, z = dz * ri;
    float tt = c.s * ri;
    // order 2
    float v2x = fmaf(c.xz, z, fmaf(c.xy, y, c.xx * x));
    float v2y = fmaf(c.yz, z, fmaf(c.yy, y, c.xy * x));
    float v2z = fmaf(c.zz, z, fmaf(c.yz, y, c.xz * x));
    float p2 = fmaf(v2z, z, fmaf(v2y, y, v2x * x));
    // order 3: quadratic monomials, cross terms carry their multiplicity 2
    float xx = x * x, yy = y * y, zz = z * z;
    float x2 = x + x, y2 = y + y;
    float xy = x2 * y, xz = x2 * z, yz = y2 * z;
    float v3x = fmaf(c.xyz, yz, fmaf(c.xxz, xz, fmaf(c.xxy, xy, fmaf(c.xzz, zz, fmaf(c.xyy, yy, c.xxx * xx)))));
    float v3y = fmaf(c.yyz, yz, fmaf(c.xyz, xz, fmaf(c.xyy, xy, fmaf(c.yzz, zz, fmaf(c.yyy, yy, c.xxy * xx)))));
    float v3z = fmaf(c.yzz, yz, fmaf(c.xzz, xz, fmaf(c.xyz, xy, fmaf(c.zzz, zz, fmaf(c.yyz, yy, c.xxz * xx)))));
    float p3 = fmaf(v3z, z, fmaf(v3y, y, v3x * x));
    // order 4: cubic monomials with multiplicities 1, 3, 6
    float x3 = 3.0f * x, y3 = 3.0f * y, z3 = 3.0f * z;
    float mxxx = xx * x, myyy = yy * y, mzzz = zz * z;
    float mxxy = xx * y3, mxxz = xx * z3, mxyy = yy * x3, myyz = yy * z3, mxzz = zz * x3, myzz = zz * y3;
    float mxyz = xy * z3;
    float v4x = fmaf(c.xzzz, mzzz, fmaf(c.xyzz, myzz, fmaf(c.xyyz, myyz, fmaf(c.xyyy, myyy, fmaf(c.xxzz, mxzz,
                fmaf(c.xxyz, mxyz, fmaf(c.xxyy, mxyy, fmaf(c.xxxz, mxxz, fmaf(c.xxxy, mxxy, c.xxxx * mxxx)))))))));
    float v4y = fmaf(c.yzzz, mzzz, fmaf(c.yyzz, myzz, fmaf(c.yyyz, myyz, fmaf(c.yyyy, myyy, fmaf(c.xyzz, mxzz,
                fmaf(c.xyyz, mxyz, fmaf(c.xyyy, mxyy, fmaf(c.xxyz, mxxz, fmaf(c.xxyy, mxxy, c.xxxy * mxxx)))))))));
    float v4z = fmaf(c.zzzz, mzzz, fmaf(c.yzzz, myzz, fmaf(c.yyzz, myyz, fmaf(c.yyyz, myyy, fmaf(c.xzzz, mxzz,
                fmaf(c.xyzz, mxyz, fmaf(c.xyyz, mxyy, fmaf(c.xxzz, mxxz, fmaf(c.xxyz, mxxy, c.xxxz * mxxx)))))))));
    float p4 = fmaf(v4z, z, fmaf(v4y, y, v4x * x));
    // combine
    float t2 = tt * tt, t3 = t2 * tt, t4 = t2 * t2;
    float e2 = t2 * p2, e3 = t3 * p3, e4 = t4 * p4;
    float fs = 1.0f + e2 + e3 + e4;                                      // potential series
    float S = fmaf(9.0f, e4, fmaf(7.0f, e3, fmaf(5.0f, e2, 1.0f)));      // radial part of the force
    float w2 = t2 + t2, w3 = 3.0f * t3, w4 = 4.0f * t4;
    float wx = fmaf(w4, v4x, fmaf(w3, v3x, w2 * v2x));
    float wy = fmaf(w4, v4y, fmaf(w3, v3y, w2 * v2y));
    float wz = fmaf(w4, v4z, fmaf(w3, v3z, w2 * v2z));
    float mr = c.M * ri;
    float mr2 = mr * ri;
    ph = fmaf(-mr, fs, ph);
    ax = fmaf(mr2, fmaf(-S, x, wx), ax);
    ay = fmaf(mr2, fmaf(-S, y, wy), ay);
    az = fmaf(mr2, fmaf(-S, z, wz), az);
}

// Butterfly transpose-reduction of NV per-lane partial sums across the 32 lanes: log2(32) rounds, in
// round with partner lane^mask each lane hands over the half of its values the partner keeps.
// NV = 64: lane l ends with the totals of values 2l, 2l+1 in v[0], v[1];  NV = 32: value l in v[0];
// NV = 16: value (l & 15) in v[0].   NV - NV/32 shuffles instead of 5 NV.
template <int NV>
__device__ __forceinline__ void warp_transpose_reduce(float (&v)[NV], int lane) {
    static_assert(NV == 16 || NV == 32 || NV == 64, "NV");
    if (NV == 16) {
#pragma unroll
        for (int i = 0; i < NV; ++i) v[i] += __shfl_xor_sync(0xffffffffu, v[i], 16);
    }
    constexpr int kFirstMask = (NV == 16) ? 8 : 16;
    int n = NV / 2;
#pragma unroll
    for (int mask = kFirstMask; mask >= 1; mask >>= 1) {
        bool up = (lane & mask) != 0;
#pragma unroll
        for (int i = 0; i < NV / 2; ++i) {
            if (i < n) {
                float send = up ? v[i] : v[i + n];
                float keep = up ? v[i + n] : v[i];
                v[i] = keep + __shfl_xor_sync(0xffffffffu, send, mask);
            }
        }
        n >>= 1;
    }
}

template <int TB, int WARPS, int MINB>
__global__ void __launch_bounds__(WARPS * 32, MINB) pkdg_eval_kernel(const EvalParams p) {
    __shared__ float4 s_tgt[WARPS][TB];
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const float4 far4 = make_float4(kFar, kFar, kFar, 0.0f);
    const bool do_pp = !(p.flags & 0x2u), do_pc = !(p.flags & 0x4u), accumulate = (p.flags & 0x1u) != 0;
    unsigned bad = 0;

    for (;;) {
        unsigned bu = 0;
        if (lane == 0) bu = atomicAdd(p.work_counter, 1u);
        bu = __shfl_sync(0xffffffffu, bu, 0);
        if ((int64_t)bu >= p.n_buckets) break;
        const BucketDesc d = p.desc[bu];
        const int pp_len = do_pp ? d.pp_len : 0, pc_len = do_pc ? d.pc_len : 0;

        for (int t0 = 0; t0 < d.count; t0 += TB) {
            const int ntp = min(TB, d.count - t0);
            __syncwarp();
            if (lane < ntp) s_tgt[warp][lane] = __ldg(p.xyzm + d.first + t0 + lane);
            __syncwarp();
            float acc[TB * 4];
#pragma unroll
            for (int i = 0; i < TB * 4; ++i) acc[i] = 0.0f;

            // ---- a3: P-P tiles; source of the next tile is in flight while this one is evaluated
            {
                const int ntile = (pp_len + 31) >> 5;
                int32_t j = ntile ? tile_entry(p.pp_idx, d.pp_begin, pp_len, 0, lane) : -1;
                if ((uint32_t)j >= (uint64_t)p.n_particles) { bad += (j >= 0); j = -1; }
                float4 s = j >= 0 ? __ldg(p.xyzm + j) : far4;
                int32_t jn = ntile > 1 ? tile_entry(p.pp_idx, d.pp_begin, pp_len, 1, lane) : -1;
                for (int k = 0; k < ntile; ++k) {
                    if ((uint32_t)jn >= (uint64_t)p.n_particles) { bad += (jn >= 0); jn = -1; }
                    const float4 sn = jn >= 0 ? __ldg(p.xyzm + jn) : far4;
                    const int32_t jnn = (k + 2 < ntile) ? tile_entry(p.pp_idx, d.pp_begin, pp_len, k + 2, lane) : -1;
                    const int self_t = j - (d.first + t0);  // sink slot this source coincides with
#pragma unroll
                    for (int t = 0; t < TB; ++t) {
                        if (t < ntp) {
                            const float4 tg = s_tgt[warp][t];
                            pp_interact(tg, s, self_t == t, p.h2min, p.hinv, acc[4 * t], acc[4 * t + 1],
                                        acc[4 * t + 2], acc[4 * t + 3]);
                        }
                    }
                    s = sn; j = jn; jn = jnn;
                }
            }
            // ---- a4: P-C tiles; the lane's cell stays in registers for all sinks of the pass
            {
                const int ntile = (pc_len + 31) >> 5;
                int32_t c = ntile ? tile_entry(p.pc_idx, d.pc_begin, pc_len, 0, lane) : -1;
                for (int k = 0; k < ntile; ++k) {
                    if ((uint32_t)c >= (uint64_t)p.n_cells) { bad += (c >= 0); c = -1; }
                    const int32_t cn = (k + 1 < ntile) ? tile_entry(p.pc_idx, d.pc_begin, pc_len, k + 1, lane) : -1;
                    CellRegs cr;
                    if (c >= 0) {
                        const float4* q = p.cellq + (int64_t)c * 8;
                        cell_unpack(cr, __ldg(q), __ldg(q + 1), __ldg(q + 2), __ldg(q + 3), __ldg(q + 4),
                                    __ldg(q + 5), __ldg(q + 6), __ldg(q + 7));
                    } else {
                        const float4 z4 = make_float4(0.f, 0.f, 0.f, 0.f);
                        cell_unpack(cr, far4, z4, z4, z4, z4, z4, z4, z4);
                    }
#pragma unroll
                    for (int t = 0; t < TB; ++t) {
                        if (t < ntp) {
                            const float4 tg = s_tgt[warp][t];
                            pc_interact(tg, cr, acc[4 * t], acc[4 * t + 1], acc[4 * t + 2], acc[4 * t + 3]);
                        }
                    }
                    c = cn;
                }
            }
            // ---- a5: cross-lane reduction and write-back
            warp_transpose_reduce<TB * 4>(acc, lane);
            float* outf = reinterpret_cast<float*>(p.out + d.first + t0);
            if (TB == 16) {
                const int t = lane >> 1;
                if (t < ntp) {
                    float2* o2 = reinterpret_cast<float2*>(outf) + lane;
                    float2 r = make_float2(acc[0], acc[1]);
                    if (accumulate) { float2 old = *o2; r.x += old.x; r.y += old.y; }
                    *o2 = r;
                }
            } else {
                const int slot = (TB == 8) ? lane : (lane & 15);
                if ((slot >> 2) < ntp && (TB == 8 || lane < 16)) {
                    float r = acc[0];
                    if (accumulate) r += outf[slot];
                    outf[slot] = r;
                }
            }
        }
    }
    if (bad) atomicAdd(&p.stats->bad_entries, (unsigned long long)bad);
}

// FFMA-only probe: 8 independent chains per thread, `iters` rounds of 8 FFMA.
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
