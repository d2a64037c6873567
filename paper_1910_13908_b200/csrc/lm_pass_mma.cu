// sagecal_lm_cost_grad_jtj for 2x2 coherencies on the FP64 tensor cores.
//
// For a fixed baseline (p, q) all T*F samples see the same J_p, J_q, so with e = vec(E), c = vec(C), x = vec(x_k) and
// W = J_p (x) conj(J_q) (vec(J_p C J_q^H) = W c) the sums of the pass are contractions over the baseline's samples:
//
//   e    = x - W c                                 per sample: (8 x 8 real)(8 x 8 samples), two DMMA per 8 samples
//   Sec  = sum_tf e c^H   (4x4 complex)            (8 x 4 samples)(4 samples x 8), two DMMA per 8 samples
//   Scc  = sum_tf c c^H   (4x4 Hermitian)          two DMMA per 8 samples
//   cost = sum_tf |e|^2
//   G_p[i,k] = sum_{j,l} J_q[j,l] Sec[(i,j),(k,l)]         G_q[j,l] = sum_{i,k} J_p[i,k] conj(Sec[(i,j),(k,l)])
//   M_p[k,k'] = sum_{l,l'} (J_q^H J_q)[l,l'] Scc[(k,l),(k',l')]     M_q[l,l'] = sum_{k,k'} (J_p^H J_p)[k,k'] conj(Scc[(k,l),(k',l')])
//
// which are E A^H, E^H T1, A A^H, T1^H T1 of the header summed over the baseline's samples (A = C J_q^H, T1 = J_p C).
// The residual e is formed per sample and the cost and Sec are taken of it directly, so nothing cancels.  One warp owns
// one baseline and walks its samples 8 at a time with the fragment layouts of wbgroup.cu (6 loads and 6 DMMA per 8
// samples, where the FMA form issues 200 FP64 instructions per sample and sits on the FP64 ridge); it leaves one
// 26-double record per baseline, and lm_reduce_mma_kernel adds each station's records in a fixed order: no atomics,
// bit-reproducible.
#include "lm_pass.cuh"

namespace sgc {

constexpr int PM_WARPS = 4;
constexpr int PM_RED_THREADS = 128;

__device__ __forceinline__ void pm_dmma(double& d0, double& d1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}
__device__ __forceinline__ int64_t pm_sample(int m, int TF, int F, int64_t B, int64_t b) {
    if (m >= TF) return -1;
    const int t = m / F;
    return ((int64_t)t * B + b) * F + (m - t * F);
}
__device__ __forceinline__ cplx pm_ld(const sagecal_c128* p) {
    const double2 v = __ldg(reinterpret_cast<const double2*>(p));
    return mk(v.x, v.y);
}

template <bool F8>
__global__ void __launch_bounds__(32 * PM_WARPS)
lm_pass_mma_kernel(int N, int T, int F, int64_t B, const sagecal_c128* __restrict__ x_, const sagecal_c128* __restrict__ coh_,
                   const sagecal_c128* __restrict__ jones, double* __restrict__ Brec) {
    __shared__ cplx s_st[PM_WARPS][32], s_cf[PM_WARPS][16];   // per warp: Sec and Scc (16 + 16), coefficients
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t b = (int64_t)blockIdx.x * PM_WARPS + warp;
    if (b >= B) return;                                   // whole warps leave together; no CTA-wide barrier below
    const int g = lane >> 2, j = lane & 3;
    const double* x = reinterpret_cast<const double*>(x_);
    const double* coh = reinterpret_cast<const double*>(coh_);
    int p, q;
    bl_stations(N, b, p, q);
    const sagecal_c128 *Jp = jones + 4 * p, *Jq = jones + 4 * q;

    // A fragments of -W, W[(i,j),(k,l)] = J_p[i,k] conj(J_q[j,l]): row g = 2a + ri, column kk = 4s + j = 2c + ri2
    double Aw[2];
    {
        const int a = g >> 1, ri = g & 1;
#pragma unroll
        for (int s = 0; s < 2; s++) {
            const int kk = 4 * s + j, c = kk >> 1, ri2 = kk & 1;
            const cplx w = cmulc(pm_ld(Jp + 2 * (a >> 1) + (c >> 1)), pm_ld(Jq + 2 * (a & 1) + (c & 1)));
            Aw[s] = -(ri == ri2 ? w.re : (ri ? w.im : -w.im));
        }
    }
    double D0 = 0.0, D1 = 0.0, S0 = 0.0, S1 = 0.0, cost = 0.0;
    const int TF = T * F;
    // (Loading the coherency samples once and transposing the 8 x 8 block with shuffles for the write-back's B fragments
    // was slower, 0.55 against 0.48 ms at cfg4: the second load hits L1.)
    auto chunk = [&](double e0, double e1, double bp0, double bp1, double bn0, double bn1) {
        pm_dmma(e0, e1, Aw[0], bp0);                     // e = x - W c
        pm_dmma(e0, e1, Aw[1], bp1);
        pm_dmma(D0, D1, e0, bn0);                        // Sec += e c^H
        pm_dmma(D0, D1, e1, bn1);
        pm_dmma(S0, S1, bn0, bn0);                       // Scc += c c^H
        pm_dmma(S0, S1, bn1, bn1);
        cost = fma(e0, e0, fma(e1, e1, cost));
    };
    if (F8) {
        // a chunk is one time slot: the lane's six offsets are fixed, the pointers advance by one slot (B*8 samples)
        const size_t slot = (size_t)B * 64;
        const double* xa = x + (size_t)b * 64 + (2 * j) * 8 + g;        // samples 2j, 2j + 1, position g
        const double* ca = coh + (size_t)b * 64 + (2 * j) * 8 + g;
        const double* cb = coh + (size_t)b * 64 + g * 8 + j;            // sample g, positions j, 4 + j
#pragma unroll 2
        for (int t = 0; t < T; t++, xa += slot, ca += slot, cb += slot)
            chunk(__ldg(xa), __ldg(xa + 8), __ldg(cb), __ldg(cb + 4), __ldg(ca), __ldg(ca + 8));
    } else {
#pragma unroll 1
        for (int m0 = 0; m0 < TF; m0 += 8) {
            const int64_t in = pm_sample(m0 + g, TF, F, B, b);
            const int64_t i0 = pm_sample(m0 + 2 * j, TF, F, B, b);
            const int64_t i1 = pm_sample(m0 + 2 * j + 1, TF, F, B, b);
            chunk(i0 >= 0 ? __ldg(x + i0 * 8 + g) : 0.0, i1 >= 0 ? __ldg(x + i1 * 8 + g) : 0.0,
                  in >= 0 ? __ldg(coh + in * 8 + j) : 0.0, in >= 0 ? __ldg(coh + in * 8 + 4 + j) : 0.0,
                  i0 >= 0 ? __ldg(coh + i0 * 8 + g) : 0.0, i1 >= 0 ? __ldg(coh + i1 * 8 + g) : 0.0);
        }
    }
    // complex entries: (rr + ii) + i (ir - ri) with the partner lane that holds the other real/imaginary row
    {
        const int a = g >> 1, ri = g & 1;
        const double p0 = __shfl_xor_sync(0xffffffffu, D0, 4), p1 = __shfl_xor_sync(0xffffffffu, D1, 4);
        const double q0 = __shfl_xor_sync(0xffffffffu, S0, 4), q1 = __shfl_xor_sync(0xffffffffu, S1, 4);
        if (ri == 0) {
            s_st[warp][4 * a + j] = mk(D0 + p1, p0 - D1);             // Sec[a][c]
            s_st[warp][16 + 4 * a + j] = mk(S0 + q1, q0 - S1);        // Scc[a][c]
        }
    }
    for (int o = 16; o > 0; o >>= 1) cost += __shfl_xor_sync(0xffffffffu, cost, o);
    // coefficients: J_q (0..3), J_p (4..7), H_q = J_q^H J_q (8..11), H_p = J_p^H J_p (12..15), row-major 2x2
    if (lane < 8) s_cf[warp][lane] = pm_ld((lane < 4 ? Jq : Jp) + (lane & 3));
    __syncwarp();
    if (lane < 8) {
        const cplx* J = s_cf[warp] + (lane & 4);
        const int u = (lane >> 1) & 1, v = lane & 1;                  // H[u,v] = sum_w conj(J[w,u]) J[w,v]
        s_cf[warp][8 + lane] = cfmaca(J[2 + u], J[2 + v], cfmaca(J[u], J[v], mk(0.0, 0.0)));
    }
    __syncwarp();
    // 14 outputs of 4 terms each, one lane per output, the same code for all:
    //   o = 0..3   G_p[i,k] = sum_{j,l} J_q[j,l]      Sec[(i,j),(k,l)]          (i, k) = (o >> 1, o & 1)
    //   o = 4..7   G_q[j,l] = sum_{i,k} J_p[i,k] conj(Sec[(i,j),(k,l)])         (j, l) = (o >> 1 & 1, o & 1)
    //   o = 8..10  M_p[r,r'] = sum_{u,v} H_q[u,v]      Scc[(r,u),(r',v)]         (r, r') = (0,0), (1,1), (0,1)
    //   o = 11..13 M_q[r,r'] = sum_{u,v} H_p[u,v] conj(Scc[(u,r),(v,r')])
    if (lane < 14) {
        const bool isM = lane >= 8;
        const int e = isM ? (lane - 8) % 3 : 0;
        const bool second = isM ? lane >= 11 : lane >= 4;             // G_q / M_q: the column station's side
        const int r = isM ? (e == 1) : ((lane >> 1) & 1), r2 = isM ? (e != 0) : (lane & 1);
        const cplx* cf = s_cf[warp] + (isM ? (second ? 12 : 8) : (second ? 4 : 0));
        const cplx* stat = s_st[warp] + (isM ? 16 : 0);
        cplx acc = mk(0.0, 0.0);
#pragma unroll
        for (int u = 0; u < 2; u++)
#pragma unroll
            for (int v = 0; v < 2; v++) {
                const int row = second ? 2 * u + r : 2 * r + u, col = second ? 2 * v + r2 : 2 * r2 + v;
                const cplx sv = stat[4 * row + col];
                acc = second ? cfmac(cf[2 * u + v], sv, acc) : cfma(cf[2 * u + v], sv, acc);
            }
        double* rec = Brec + (size_t)b * PASS_BREC;
        if (!isM) { rec[2 * lane] = acc.re; rec[2 * lane + 1] = acc.im; }
        else {
            const int base = second ? 20 : 16;
            if (e < 2) rec[base + e] = acc.re;
            else { rec[base + 2] = acc.re; rec[base + 3] = acc.im; }
        }
    } else if (lane == 14) {
        double* rec = Brec + (size_t)b * PASS_BREC;
        rec[24] = cost;
        rec[25] = 0.0;
    }
}

// block s: station s adds its N - 1 records in a fixed order (as column station of (p, s), p < s, then as row station
// of (s, q), q > s) and the cost of its row-role records (every baseline is the row-role record of exactly one
// station).  The block that finishes last (integer ticket counter, control flow only) adds the N partial costs, again in
// a fixed order, and re-arms the counter.
__global__ void __launch_bounds__(PM_RED_THREADS)
lm_reduce_mma_kernel(int N, const double* __restrict__ Brec, double* __restrict__ cost_st, unsigned* counter,
                     double* __restrict__ cost, sagecal_c128* __restrict__ grad, sagecal_c128* __restrict__ jtj) {
    constexpr int NV = PASS_NV + 1;
    __shared__ double s_red[NV][PM_RED_THREADS];
    __shared__ bool s_last;
    const int tid = threadIdx.x, s = blockIdx.x;
    double acc[NV];
#pragma unroll
    for (int i = 0; i < NV; i++) acc[i] = 0.0;
    for (int e = tid; e < N - 1; e += PM_RED_THREADS) {
        const bool colrole = e < s;
        const int64_t b = colrole ? bl_index(N, e, s) : bl_index(N, s, e + 1);
        const double2* rec = reinterpret_cast<const double2*>(Brec + (size_t)b * PASS_BREC);
        const double2* gsrc = rec + (colrole ? 4 : 0);
        const double2* msrc = rec + (colrole ? 10 : 8);
#pragma unroll
        for (int i = 0; i < 4; i++) { const double2 v = __ldcg(gsrc + i); acc[2 * i] += v.x; acc[2 * i + 1] += v.y; }
#pragma unroll
        for (int i = 0; i < 2; i++) { const double2 v = __ldcg(msrc + i); acc[8 + 2 * i] += v.x; acc[9 + 2 * i] += v.y; }
        if (!colrole) acc[PASS_NV] += __ldcg(rec + 12).x;
    }
    auto block_sum = [&]() {
#pragma unroll
        for (int i = 0; i < NV; i++) s_red[i][tid] = acc[i];
        __syncthreads();
        for (int o = PM_RED_THREADS / 2; o > 0; o >>= 1) {
            if (tid < o) {
#pragma unroll
                for (int i = 0; i < NV; i++) s_red[i][tid] += s_red[i][tid + o];
            }
            __syncthreads();
        }
    };
    block_sum();
    if (tid == 0) {
        sagecal_c128* G = grad + (size_t)s * 4;
        sagecal_c128* M = jtj + (size_t)s * 4;
        for (int i = 0; i < 4; i++) { G[i].re = s_red[2 * i][0]; G[i].im = s_red[2 * i + 1][0]; }
        M[0].re = s_red[8][0];  M[0].im = 0.0;
        M[1].re = s_red[10][0]; M[1].im = s_red[11][0];
        M[2].re = s_red[10][0]; M[2].im = -s_red[11][0];
        M[3].re = s_red[9][0];  M[3].im = 0.0;
        cost_st[s] = s_red[PASS_NV][0];
        __threadfence();
        s_last = atomicAdd(counter, 1u) == (unsigned)(N - 1);
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
#pragma unroll
    for (int i = 0; i < NV; i++) acc[i] = 0.0;
    for (int e = tid; e < N; e += PM_RED_THREADS) acc[0] += __ldcg(cost_st + e);
    __syncthreads();
    block_sum();
    if (tid == 0) {
        *cost = s_red[0][0];
        *counter = 0u;
    }
}

int enqueue_pass_mma(const PassGeom& g, const PassWorkspace& w, const sagecal_c128* x, const sagecal_c128* coh_k,
                     const sagecal_c128* jones, double* cost, sagecal_c128* grad, sagecal_c128* jtj, cudaStream_t st) {
    {
        LaunchScope ls(KK_PASS, st);
        const unsigned grid = (unsigned)((g.B + PM_WARPS - 1) / PM_WARPS);
        if (g.F == 8) lm_pass_mma_kernel<true><<<grid, 32 * PM_WARPS, 0, st>>>(g.N, g.T, g.F, g.B, x, coh_k, jones, w.Brec);
        else lm_pass_mma_kernel<false><<<grid, 32 * PM_WARPS, 0, st>>>(g.N, g.T, g.F, g.B, x, coh_k, jones, w.Brec);
        SGC_LAUNCH_CHECK();
    }
    SGC_CUDA(cudaMemsetAsync(w.counter, 0, sizeof(unsigned), st));   // caller's workspace: contents unknown
    {
        LaunchScope ls(KK_REDUCE, st);
        lm_reduce_mma_kernel<<<g.N, PM_RED_THREADS, 0, st>>>(g.N, w.Brec, w.cost_st, w.counter, cost, grad, jtj);
        SGC_LAUNCH_CHECK();
    }
    return SAGECAL_OK;
}

}  // namespace sgc
