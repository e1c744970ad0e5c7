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
// lists; a lane keeps its partial sums of the local coefficients in registers across both lists.  Everything is
// made dimensionless with ONE length per bucket, lambda = max_i |x_i - z_B|: the lane accumulates
// lambda^|n| n! L_n from D_k lambda^|k| = (lambda/|R|)^|k| / |R| x (polynomial in the unit vector R/|R|) and
// moments divided by lambda^|m|, so no intermediate leaves the fp32 range for any |R| and the sinks evaluate a
// polynomial in sigma = s / lambda, |sigma| <= 1.  1/|R| is harmonic, so only the 36 coefficients with at most one
// z index are accumulated, from 22 folded moments per cell (gen_fmm.py "Trace-free"): 215 multiply-adds per cell
// instead of 336, 128 registers and 16 warps per SM instead of 255 and 8; the other 20 coefficients are rebuilt once
// per bucket.  The derivative polynomials, the moment folding and the shift are generated straight-line code
// (pkdg_fmm_gen.cuh, written by gen_fmm.py from the definition of D_k by exact differentiation -- not from a
// recurrence).  The 32 lane partials of each coefficient are summed through shared memory in a fixed order, then
// lanes = sinks evaluate the polynomial and its gradient.
// Flops as executed (add / mul = 1, FMA = 2, rsqrt = 1): per C-C entry 23 (geometry, Newton step) + 52 (monomials)
// + 224 (derivative polynomials: 112 terms, 46 scalings) + 86 (folded moments: 43 terms, 22 scalings) + 430 (shift:
// 215 FMA) = 815; per C-P entry 23 + 52 + 224 + 73 = 372; per sink 6 + 52 + 112 + 315 + 3 = 488; per bucket 1488
// (reduction of 36 x 32 partials, rebuilding the 56).  The paper's audit of its own CPU code gives 472 + rsqrt /
// 206 + rsqrt (Table 3).
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

// Per-warp shared memory: while the source lists are walked it holds the lane's NEXT cell record (cp.async, two
// buffers of 9 x 16 bytes per lane, [buffer][part][lane]: conflict-free) -- a lane needs ~800 clocks for one C-C
// entry and two warps per scheduler cannot hide a global load behind that; afterwards the same bytes hold the
// 32 lane partials of the 56 coefficients for the reduction.
constexpr int kFmmStageF4 = 2 * 9 * 32;                                        // float4 per warp
constexpr int kFmmWarpFloats = kFmmStageF4 * 4 > kNLoc * kFmmRow ? kFmmStageF4 * 4 : kNLoc * kFmmRow;

// What is fetched ahead for a bucket, in three dependent steps (A: its ranges, B: the first list entries and the
// lane's sink, C: the first sources), each issued one phase of arithmetic before the next needs it: a bucket has only
// ~3 + 2 trips over its lists, so without this seven dependent global loads would sit in front of ~4000 clocks of
// arithmetic and two warps per scheduler cannot hide them.
struct FmmAhead {
    unsigned bu;
    int first, count;
    float zx, zy, zz;
    int64_t cc0, cc1, cp0, cp1;
    int32_t icc0, icc1, jcp0, jcp1;   // first list entries of the lane, as loaded (validated when they are used)
    float4 sink, pcp0;
};

__global__ void __launch_bounds__(kFmmWarps * 32, 4) pkdg_fmm_kernel(const FmmParams p) {
    __shared__ __align__(16) float s_part[kFmmWarps][kFmmWarpFloats];
    __shared__ float s_lam[kFmmWarps][64];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    float* part = s_part[warp];
    float4* stage = reinterpret_cast<float4*>(s_part[warp]);
    float* Lam = s_lam[warp];
    const bool accumulate = (p.flags & 0x1u) != 0;
    unsigned long long n_cc = 0, n_cp = 0, bad = 0;   // lane 0 counts list lengths, every lane its bad entries

    // Entry e of a list as it is stored (-1 beyond the end).  Nothing looks at the value here: a load whose result is
    // tested at once stalls the warp for the whole memory latency; cc_valid / cp_valid test it one trip later.
    auto cc_entry = [&](const FmmAhead& m, int64_t e) -> int32_t { return e < m.cc1 ? __ldg(p.cc_idx + e) : -1; };
    auto cp_entry = [&](const FmmAhead& m, int64_t e) -> int32_t { return e < m.cp1 ? __ldg(p.cp_idx + e) : -1; };
    auto cc_valid = [&](int32_t c) -> int32_t {
        if (c >= 0 && (int64_t)c >= p.n_cells) { ++bad; return -1; }
        return c;
    };
    auto cp_valid = [&](int32_t j) -> int32_t {
        if (j >= 0 && (int64_t)j >= p.n_particles) { ++bad; return -1; }
        return j;
    };
    auto issue_rec = [&](int32_t c, int buf) {   // rec_vec4: records are 16-byte aligned with a stride that keeps them so
        if (c >= 0 && p.rec_vec4) {
            const float4* r4 = reinterpret_cast<const float4*>(p.rec + (int64_t)c * p.stride);
#pragma unroll
            for (int i = 0; i < 9; ++i) cp_async16(stage + (buf * 9 + i) * 32 + lane, r4 + i);
        }
        cp_async_commit();
    };
    auto step_a = [&](FmmAhead& m) {   // needs m.bu
        const int64_t b = m.bu;
        m.first = __ldg(p.first + b); m.count = __ldg(p.count + b);
        m.zx = __ldg(p.centre + 3 * b); m.zy = __ldg(p.centre + 3 * b + 1); m.zz = __ldg(p.centre + 3 * b + 2);
        m.cc0 = m.cc1 = m.cp0 = m.cp1 = 0;
        if (p.cc_off) { m.cc0 = __ldg(p.cc_off + b); m.cc1 = __ldg(p.cc_off + b + 1); }
        if (p.cp_off) { m.cp0 = __ldg(p.cp_off + b); m.cp1 = __ldg(p.cp_off + b + 1); }
    };
    auto step_b = [&](FmmAhead& m) {   // needs step A
        if (m.count < 0 || m.first < 0 || (int64_t)m.first + m.count > p.n_particles) { bad += (lane == 0); m.count = 0; }
        if (m.cc1 < m.cc0) { bad += (lane == 0); m.cc1 = m.cc0; }
        if (m.cp1 < m.cp0) { bad += (lane == 0); m.cp1 = m.cp0; }
        m.icc0 = cc_entry(m, m.cc0 + lane); m.icc1 = cc_entry(m, m.cc0 + lane + 32);
        m.jcp0 = cp_entry(m, m.cp0 + lane); m.jcp1 = cp_entry(m, m.cp0 + lane + 32);
        m.sink = lane < m.count ? __ldg(p.xyzm + m.first + lane) : make_float4(m.zx, m.zy, m.zz, 0.0f);
    };
    auto step_c = [&](FmmAhead& m) {   // needs step B; the staging memory must be free
        m.icc0 = cc_valid(m.icc0);
        issue_rec(m.icc0, 0);
        m.jcp0 = cp_valid(m.jcp0);
        m.pcp0 = m.jcp0 >= 0 ? __ldg(p.xyzm + m.jcp0) : make_float4(0.f, 0.f, 0.f, 0.f);
    };
    auto claim = [&]() -> unsigned {
        unsigned v = 0;
        if (lane == 0) v = atomicAdd(p.work_counter, 1u);
        return v;
    };

    FmmAhead cur;
    cur.bu = __shfl_sync(0xffffffffu, claim(), 0);
    if ((int64_t)cur.bu >= p.n_buckets) return;
    step_a(cur); step_b(cur); step_c(cur);
    unsigned claimed = claim();   // buckets are claimed one iteration before they are looked at

    for (;;) {
        FmmAhead nxt;
        nxt.bu = __shfl_sync(0xffffffffu, claimed, 0);
        claimed = claim();
        const int first = cur.first, count = cur.count;
        const float zx = cur.zx, zy = cur.zy, zz = cur.zz;

        // lambda = the largest distance of a sink from the centre (1 if the bucket is a point at its centre)
        float lam2;
        {
            const float sx = cur.sink.x - zx, sy = cur.sink.y - zy, sz = cur.sink.z - zz;
            lam2 = fmaf(sz, sz, fmaf(sy, sy, sx * sx));
        }
        for (int t = lane + 32; t < count; t += 32) {
            const float4 x = __ldg(p.xyzm + first + t);
            const float sx = x.x - zx, sy = x.y - zy, sz = x.z - zz;
            lam2 = fmaxf(lam2, fmaf(sz, sz, fmaf(sy, sy, sx * sx)));
        }
#pragma unroll
        for (int o = 16; o; o >>= 1) lam2 = fmaxf(lam2, __shfl_xor_sync(0xffffffffu, lam2, o));
        const float lam = lam2 > 0.0f ? sqrtf(lam2) : 1.0f;
        const float il = 1.0f / lam;

        const bool has_next = (int64_t)nxt.bu < p.n_buckets;
        if (has_next) step_a(nxt);

        float L[kNRed];   // the 36 coefficients with at most one z; the other 20 follow from them (1/|R| is harmonic)
#pragma unroll
        for (int i = 0; i < kNRed; ++i) L[i] = 0.0f;

        // ---- C-C: one source cell per lane and trip; the record of trip t + 1 and the index of trip t + 2 are in
        //      flight during trip t (the record of trip 0 since step C)
        if (p.cc_off) {
            const int64_t e0 = cur.cc0, e1 = cur.cc1;
            if (lane == 0) n_cc += (unsigned long long)(e1 - e0);
            // -(-1)^|m| / lambda^|m| for |m| = 0, 2, 3, 4
            const float il2 = il * il;
            const float sc0 = -1.0f, sc2 = -il2, sc3 = il2 * il, sc4 = -il2 * il2;
            int32_t c_cur = cur.icc0, c_nxt = cur.icc1;
            int buf = 0;
#pragma unroll 1
            for (int64_t e = e0; e < e1; e += 32) {   // warp-uniform trips
                const int32_t c = c_cur;
                c_cur = cc_valid(c_nxt);
                issue_rec(c_cur, buf ^ 1);
                c_nxt = cc_entry(cur, e + lane + 64);
                cp_async_wait_pending<1>();            // this trip's record has landed (only the lane itself reads it)
                const int bsel = buf;
                buf ^= 1;
                if (c < 0) continue;                   // padding, bad entry, or past the end of the list
                float q[36];
                if (p.rec_vec4) {
#pragma unroll
                    for (int i = 0; i < 9; ++i) {
                        const float4 v = stage[(bsel * 9 + i) * 32 + lane];
                        q[4 * i] = v.x; q[4 * i + 1] = v.y; q[4 * i + 2] = v.z; q[4 * i + 3] = v.w;
                    }
                } else {
                    const float* r = p.rec + (int64_t)c * p.stride;
#pragma unroll
                    for (int i = 0; i < 35; ++i) q[i] = __ldg(r + i);
                }
                float d[kNLoc];
                fmm_source_derivs(zx - q[0], zy - q[1], zz - q[2], lam, d);
                float F[kNFold];
                fmm_fold_moments(q, sc0, sc2, sc3, sc4, F);
                fmm_m2l_cell(d, F, L);
            }
        }
        cp_async_wait_all();
        if (has_next) step_b(nxt);

        // ---- C-P: one source particle per lane and trip; the particle of the next trip is loaded before this trip's
        //      arithmetic (the one of trip 0 since step C)
        if (p.cp_off) {
            const int64_t e0 = cur.cp0, e1 = cur.cp1;
            if (lane == 0) n_cp += (unsigned long long)(e1 - e0);
            float4 s_cur = cur.pcp0;
            bool ok_cur = cur.jcp0 >= 0;
            int32_t j_nxt = cur.jcp1;   // index of trip t + 1 (loaded a trip ago), particle of trip t + 1 loaded now
#pragma unroll 1
            for (int64_t e = e0; e < e1; e += 32) {
                const int32_t jn = cp_valid(j_nxt);
                const float4 s_nxt = jn >= 0 ? __ldg(p.xyzm + jn) : make_float4(0.f, 0.f, 0.f, 0.f);
                j_nxt = cp_entry(cur, e + lane + 64);
                if (ok_cur) {
                    float d[kNLoc];
                    fmm_source_derivs(zx - s_cur.x, zy - s_cur.y, zz - s_cur.z, lam, d);
                    fmm_m2l_particle(d, -s_cur.w, L);
                }
                s_cur = s_nxt; ok_cur = jn >= 0;
            }
        }

        // ---- the 32 lane partials of each accumulated coefficient, summed in a fixed order; then all 56 coefficients
        //      from the 36 (full[k + 2ez] = -full[k + 2ex] - full[k + 2ey], as a table) and 1 / n!
        __syncwarp();
#pragma unroll
        for (int i = 0; i < kNRed; ++i) part[i * kFmmRow + lane] = L[i];
        __syncwarp();
        float red0 = 0.0f, red1 = 0.0f;
#pragma unroll 8
        for (int j = 0; j < 32; ++j) red0 += part[lane * kFmmRow + j];
        if (lane + 32 < kNRed) {
#pragma unroll 8
            for (int j = 0; j < 32; ++j) red1 += part[(lane + 32) * kFmmRow + j];
        }
        __syncwarp();
        part[lane] = red0;                       // the reduced coefficients, in the first floats of the same memory
        if (lane + 32 < kNRed) part[lane + 32] = red1;
        __syncwarp();
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int i = lane + 32 * h;
            if (i < kNLoc) {
                const float full = kExpCoef[i][0] * part[kExpIdx[i][0]] + kExpCoef[i][1] * part[kExpIdx[i][1]] +
                                   kExpCoef[i][2] * part[kExpIdx[i][2]];
                Lam[i] = full * kLocInvFact[i];
            }
        }
        __syncwarp();   // the staging memory is free again, Lam is visible
        if (has_next) step_c(nxt);

        // ---- lanes = sinks: the polynomial in sigma = s / lambda and its gradient
        for (int t = lane; t < count; t += 32) {
            const float4 x = t == lane ? cur.sink : __ldg(p.xyzm + first + t);
            float m[kNLoc];
            fmm_monomials((x.x - zx) * il, (x.y - zy) * il, (x.z - zz) * il, m);
            float phi, gx, gy, gz;
            fmm_eval(m, Lam, phi, gx, gy, gz);
            float4 r = make_float4(-gx * il, -gy * il, -gz * il, phi);
            if (accumulate) { const float4 o = p.out[first + t]; r.x += o.x; r.y += o.y; r.z += o.z; r.w += o.w; }
            p.out[first + t] = r;
        }
        if (!has_next) break;
        __syncwarp();   // Lam is rewritten by the next bucket only after every lane has evaluated its sinks
        cur = nxt;
    }
    cp_async_wait_all();
    n_cc = warp_sum_u64(n_cc); n_cp = warp_sum_u64(n_cp); bad = warp_sum_u64(bad);
    if (lane == 0) {
        if (n_cc) atomicAdd(&p.stats->interactions_cc, n_cc);
        if (n_cp) atomicAdd(&p.stats->interactions_cp, n_cp);
        if (bad) atomicAdd(&p.stats->bad_entries, bad);
    }
}

}  // namespace pkdg
