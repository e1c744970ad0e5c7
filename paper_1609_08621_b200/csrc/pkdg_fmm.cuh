// pkdg_fmm.cuh -- cell-cell / cell-particle interactions and the 5th-order local expansion
// ("FMM also considers cell-cell (CC) interactions by approximating the
// potential landscape within a given cell (the sink cell) that is induced by a sufficiently distant multipole
// (the source cell)"; L69 fn 2 cell-particle interactions; L71 "The local expansion of the potential about the
// sink's center of mass is actually done to 5th order ... accumulating the CC and CP interactions").
//
// What is computed (readings A20-A22).  Sink bucket B with centre z_B; source cell C with centre z_C and
// raw moments M_m (|m| in {0, 2, 3, 4}), or source particle (x_j, m_j) = a cell with only M_0.  With
// R = z_B - z_C and D_k(R) = d^k (1/|R|):
//     L_n  = -(1/n!) sum_m (-1)^|m| (M_m / m!) D_{n+m}(R),   |n| <= 5,  |n| + |m| <= 5
//     phi(x_i) += sum_n L_n s^n,   a(x_i) -= grad of that polynomial,   s = x_i - z_B.
//
// Mapping.  One warp per sink bucket (buckets from an atomic counter, tree order).  Lanes stride the two source
// lists; a lane keeps its partial sum of the 56 coefficients in registers across both lists.  Everything is
// made dimensionless with ONE length per bucket, lambda = max_i |x_i - z_B|: the lane accumulates
// lambda^|n| n! L_n from D_k lambda^|k| = (lambda/|R|)^|k| / |R| x (polynomial in the unit vector R/|R|) and
// moments divided by lambda^|m|, so no intermediate leaves the fp32 range for any |R| and the sinks evaluate a
// polynomial in sigma = s / lambda, |sigma| <= 1.  The derivative polynomials and the 336 multiply-adds of the
// shift are generated straight-line code (pkdg_fmm_gen.cuh, written by gen_fmm.py from the definition of D_k by
// exact differentiation -- not from a recurrence).  The 32 lane partials of each coefficient are summed through
// shared memory in a fixed order, then lanes = sinks evaluate the polynomial and its gradient.
// Flops as executed (add / mul = 1, FMA = 2, rsqrt = 1): per C-C entry 23 (geometry, Newton step) + 52 (monomials)
// + 280 (derivative polynomials: 140 terms, 56 scalings) + 64 (moments) + 672 (shift: 336 FMA) = 1091; per C-P entry
// 23 + 52 + 280 + 113 = 468; per sink 6 + 52 + 112 + 315 + 3 = 488; per bucket 1848 (reduction).  The paper's
// audit of its own CPU code gives 472 + rsqrt / 206 + rsqrt (Table 3).
#pragma once
#include "pkdg_fmm_gen.cuh"

namespace pkdg {

struct FmmParams {
    const float4* xyzm;
    const float* rec;       // canonical cell records
    int32_t stride;
    int32_t rec_vec4;       // records are 16-byte aligned: float4 loads
    int64_t n_particles, n_cells, n_buckets;
    const int32_t* first;
    const int32_t* count;
    const float* centre;    // [n_buckets][3]: centre of the local expansion of each bucket
    const int64_t* cc_off;  // NULL = no list of this kind
    const int32_t* cc_idx;
    const int64_t* cp_off;
    const int32_t* cp_idx;
    float4* out;
    DevStats* stats;
    unsigned int* work_counter;
    uint32_t flags;
};

constexpr int kFmmWarps = 4;
constexpr int kFmmRow = 33;   // row stride of the per-warp reduction buffer: conflict-free both ways

// Geometry of one source seen from the sink centre: unit vector monomials -> scaled derivative tensors.
__device__ __forceinline__ void fmm_source_derivs(const float Rx, const float Ry, const float Rz, const float lam,
                                                  float (&d)[kNLoc]) {
    const float r2 = fmaf(Rz, Rz, fmaf(Ry, Ry, Rx * Rx));
    float ri = rsqrt_approx(r2);
    ri = ri * fmaf(-0.5f * r2, ri * ri, 1.5f);   // one Newton step: L_0 and L_1 carry 1/|R| and 1/|R|^3 undamped
    const float gam = lam * ri;
    float g[6];
    g[0] = ri;
#pragma unroll
    for (int n = 1; n < 6; ++n) g[n] = g[n - 1] * gam;
    float p[kNLoc];
    fmm_monomials(Rx * ri, Ry * ri, Rz * ri, p);
    fmm_derivs(p, g, d);
}

__global__ void __launch_bounds__(kFmmWarps * 32, 2) pkdg_fmm_kernel(const FmmParams p) {
    __shared__ float s_part[kFmmWarps][kNLoc * kFmmRow];
    __shared__ float s_lam[kFmmWarps][64];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    float* part = s_part[warp];
    float* Lam = s_lam[warp];
    const bool accumulate = (p.flags & 0x1u) != 0;
    unsigned long long n_cc = 0, n_cp = 0, bad = 0;   // lane 0 counts list lengths, every lane its bad entries

    for (;;) {
        unsigned bu = 0;
        if (lane == 0) bu = atomicAdd(p.work_counter, 1u);
        bu = __shfl_sync(0xffffffffu, bu, 0);
        if ((int64_t)bu >= p.n_buckets) break;
        const int64_t b = bu;
        int first = __ldg(p.first + b), count = __ldg(p.count + b);
        if (count < 0 || first < 0 || (int64_t)first + count > p.n_particles) { bad += (lane == 0); count = 0; }
        const float zx = __ldg(p.centre + 3 * b), zy = __ldg(p.centre + 3 * b + 1), zz = __ldg(p.centre + 3 * b + 2);

        // lambda = the largest distance of a sink from the centre (1 if the bucket is a point at its centre)
        float lam2 = 0.0f;
        for (int t = lane; t < count; t += 32) {
            const float4 x = __ldg(p.xyzm + first + t);
            const float sx = x.x - zx, sy = x.y - zy, sz = x.z - zz;
            lam2 = fmaxf(lam2, fmaf(sz, sz, fmaf(sy, sy, sx * sx)));
        }
#pragma unroll
        for (int o = 16; o; o >>= 1) lam2 = fmaxf(lam2, __shfl_xor_sync(0xffffffffu, lam2, o));
        const float lam = lam2 > 0.0f ? sqrtf(lam2) : 1.0f;
        const float il = 1.0f / lam;

        float L[kNLoc];
#pragma unroll
        for (int i = 0; i < kNLoc; ++i) L[i] = 0.0f;

        // ---- C-C: one source cell per lane and trip
        if (p.cc_off) {
            int64_t e0 = __ldg(p.cc_off + b), e1 = __ldg(p.cc_off + b + 1);
            if (e1 < e0) { bad += (lane == 0); e1 = e0; }
            if (lane == 0) n_cc += (unsigned long long)(e1 - e0);
            // -(-1)^|m| / lambda^|m| for |m| = 0, 2, 3, 4
            const float il2 = il * il;
            const float sc0 = -1.0f, sc2 = -il2, sc3 = il2 * il, sc4 = -il2 * il2;
#pragma unroll 1
            for (int64_t e = e0 + lane; e < e1; e += 32) {
                const int32_t c = __ldg(p.cc_idx + e);
                if (c < 0) continue;                                   // padding
                if ((int64_t)c >= p.n_cells) { ++bad; continue; }
                const float* r = p.rec + (int64_t)c * p.stride;
                float q[36];
                if (p.rec_vec4) {
                    const float4* r4 = reinterpret_cast<const float4*>(r);
#pragma unroll
                    for (int i = 0; i < 9; ++i) {
                        const float4 v = __ldg(r4 + i);
                        q[4 * i] = v.x; q[4 * i + 1] = v.y; q[4 * i + 2] = v.z; q[4 * i + 3] = v.w;
                    }
                } else {
#pragma unroll
                    for (int i = 0; i < 35; ++i) q[i] = __ldg(r + i);
                }
                float d[kNLoc];
                fmm_source_derivs(zx - q[0], zy - q[1], zz - q[2], lam, d);
                float mu[32];
#pragma unroll
                for (int s = 0; s < 32; ++s) {
                    const float sc = kMuOrder[s] == 0 ? sc0 : kMuOrder[s] == 2 ? sc2 : kMuOrder[s] == 3 ? sc3 : sc4;
                    mu[s] = (q[kMuRec[s]] * kMuInvFact[s]) * sc;
                }
                fmm_m2l_cell(d, mu, L);
            }
        }
        // ---- C-P: one source particle per lane and trip
        if (p.cp_off) {
            int64_t e0 = __ldg(p.cp_off + b), e1 = __ldg(p.cp_off + b + 1);
            if (e1 < e0) { bad += (lane == 0); e1 = e0; }
            if (lane == 0) n_cp += (unsigned long long)(e1 - e0);
#pragma unroll 1
            for (int64_t e = e0 + lane; e < e1; e += 32) {
                const int32_t j = __ldg(p.cp_idx + e);
                if (j < 0) continue;
                if ((int64_t)j >= p.n_particles) { ++bad; continue; }
                const float4 s = __ldg(p.xyzm + j);
                float d[kNLoc];
                fmm_source_derivs(zx - s.x, zy - s.y, zz - s.z, lam, d);
                fmm_m2l_particle(d, -s.w, L);
            }
        }

        // ---- the 32 lane partials of each coefficient, summed in a fixed order; 1 / n!
        __syncwarp();
#pragma unroll
        for (int i = 0; i < kNLoc; ++i) part[i * kFmmRow + lane] = L[i];
        __syncwarp();
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int i = lane + 32 * h;
            if (i < kNLoc) {
                float sum = 0.0f;
#pragma unroll 8
                for (int j = 0; j < 32; ++j) sum += part[i * kFmmRow + j];
                Lam[i] = sum * kLocInvFact[i];
            }
        }
        __syncwarp();

        // ---- lanes = sinks: the polynomial in sigma = s / lambda and its gradient
        for (int t = lane; t < count; t += 32) {
            const float4 x = __ldg(p.xyzm + first + t);
            float m[kNLoc];
            fmm_monomials((x.x - zx) * il, (x.y - zy) * il, (x.z - zz) * il, m);
            float phi, gx, gy, gz;
            fmm_eval(m, Lam, phi, gx, gy, gz);
            float4 r = make_float4(-gx * il, -gy * il, -gz * il, phi);
            if (accumulate) { const float4 o = p.out[first + t]; r.x += o.x; r.y += o.y; r.z += o.z; r.w += o.w; }
            p.out[first + t] = r;
        }
    }
    n_cc = warp_sum_u64(n_cc); n_cp = warp_sum_u64(n_cp); bad = warp_sum_u64(bad);
    if (lane == 0) {
        if (n_cc) atomicAdd(&p.stats->interactions_cc, n_cc);
        if (n_cp) atomicAdd(&p.stats->interactions_cp, n_cp);
        if (bad) atomicAdd(&p.stats->bad_entries, bad);
    }
}

}  // namespace pkdg
