// sagecal_lm_cost_grad_jtj: fused cost + gradient + per-station J^H J pass for one cluster
// (DESIGN.md §5.3).
//
//   E = x - J_p C J_q^H;  cost = sum ||E||^2;  G_p += E A^H, G_q += E^H T1;  M_p += A A^H, M_q += T1^H T1
//   with T1 = J_p C, A = C J_q^H.
//
// HBM-bound streaming pass.  No global atomics: a thread accumulates its baseline's contributions in registers
// over the time/channel loop; the row-station (p) side is reduced per unit with warp shuffles, the column-station
// (q) side stays in registers for a whole column tile and is flushed once; a second small kernel adds the
// partials per station in a fixed order, so results are bit-reproducible.
#include "lm_pass.cuh"

namespace sgc {

// ---- geometry -------------------------------------------------------------------------------------------------
PassGeom make_pass_geom(int N, int T, int F) {
    PassGeom g;
    g.N = N; g.T = T; g.F = F;
    g.TQ = F >= PASS_THREADS ? 1 : PASS_THREADS / F;
    g.nchunk = (g.TQ * F + PASS_THREADS - 1) / PASS_THREADS;
    g.ncols = (N + g.TQ - 1) / g.TQ;
    g.B = (int64_t)N * (N - 1) / 2;
    g.R = g.cum(g.ncols - 1) + (N - 1);
    g.nslots = num_sms() * 3;
    // enough units per CTA for an even static split: aim for >= 8 per slot, by cutting rows along time
    int64_t want = 8LL * g.nslots;
    int tc = (int)((want + g.R - 1) / g.R);
    if (tc < 1) tc = 1;
    if (tc > T) tc = T;
    g.tlen = (T + tc - 1) / tc;
    g.TC = (T + g.tlen - 1) / g.tlen;
    g.U = g.R * g.TC;
    if (g.nslots > g.U) g.nslots = (int)g.U;
    return g;
}

size_t pass_workspace_bytes(const PassGeom& g) {
    size_t n = 0;
    n += round_up(sizeof(double) * (size_t)g.U * PASS_WARPS * PASS_NV, 256);
    n += round_up(sizeof(double) * (size_t)g.U * PASS_WARPS, 256);
    n += round_up(sizeof(double) * (size_t)(g.nslots + g.ncols) * g.TQ * PASS_NV, 256);
    n += round_up(sizeof(double) * (size_t)g.B * PASS_BREC, 256);
    n += round_up(sizeof(double) * (size_t)g.N, 256) + 256;
    return n;
}

PassWorkspace carve_pass_workspace(const PassGeom& g, void* ws) {
    PassWorkspace w;
    char* p = (char*)ws;
    w.Ppart = (double*)p; p += round_up(sizeof(double) * (size_t)g.U * PASS_WARPS * PASS_NV, 256);
    w.Pcost = (double*)p; p += round_up(sizeof(double) * (size_t)g.U * PASS_WARPS, 256);
    w.Qpart = (double*)p; p += round_up(sizeof(double) * (size_t)(g.nslots + g.ncols) * g.TQ * PASS_NV, 256);
    w.Brec = (double*)p; p += round_up(sizeof(double) * (size_t)g.B * PASS_BREC, 256);
    w.cost_st = (double*)p; p += round_up(sizeof(double) * (size_t)g.N, 256);
    w.counter = (unsigned*)p;
    return w;
}

// ---- per-thread accumulators ----------------------------------------------------------------------------------
struct Side {               // one station side: G (2x2 complex) and Hermitian M
    cplx G[4];
    double M00, M11;
    cplx M01;
    __device__ __forceinline__ void zero() {
        G[0] = G[1] = G[2] = G[3] = M01 = mk(0.0, 0.0);
        M00 = M11 = 0.0;
    }
    __device__ __forceinline__ double get(int i) const {
        switch (i) {
            case 0: return G[0].re; case 1: return G[0].im; case 2: return G[1].re; case 3: return G[1].im;
            case 4: return G[2].re; case 5: return G[2].im; case 6: return G[3].re; case 7: return G[3].im;
            case 8: return M00; case 9: return M11; case 10: return M01.re; default: return M01.im;
        }
    }
};

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// H = J^H J as (H00, H11, H01)
__device__ __forceinline__ void gram(const m22& J, double& h00, double& h11, cplx& h01) {
    h00 = cabs2(J.a[2], cabs2(J.a[0], 0.0));
    h11 = cabs2(J.a[3], cabs2(J.a[1], 0.0));
    h01 = cfmaca(J.a[2], J.a[3], cfmaca(J.a[0], J.a[1], mk(0.0, 0.0)));
}

// Scalar coherencies (C = c I2).  General 2x2 coherencies take the tensor-core form in lm_pass_mma.cu.
__global__ void __launch_bounds__(PASS_THREADS, 3)
lm_pass_scalar_kernel(PassGeom g, const sagecal_c128* __restrict__ x, const sagecal_c128* __restrict__ coh,
               const sagecal_c128* __restrict__ jones, double* __restrict__ Ppart, double* __restrict__ Pcost,
               double* __restrict__ Qpart) {
    __shared__ double s_red[PASS_NV][PASS_THREADS];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int slot_id = blockIdx.x;
    const int64_t u_begin = g.slot_begin(slot_id), u_end = g.slot_begin(slot_id + 1);
    const int F = g.F, TQ = g.TQ, N = g.N;
    const int nper = g.nchunk > 1 ? PASS_THREADS : F;        // threads that share one q
    const int ql = g.nchunk > 1 ? 0 : tid / F;               // my column-local station
    const bool thread_used = g.nchunk > 1 ? true : tid < TQ * F;

    int cur_c = -1, cur_p = -1, q = 0;
    m22 Jp, Jq;
    double hq00 = 0, hq11 = 0, hp00 = 0, hp11 = 0;
    cplx hq01 = mk(0, 0), hp01 = mk(0, 0);
    Side sq;
    sq.zero();

    auto flush_q = [&](int c) {
        __syncthreads();
#pragma unroll
        for (int i = 0; i < PASS_NV; i++) s_red[i][tid] = sq.get(i);
        __syncthreads();
        double* out = Qpart + (size_t)(slot_id + c) * TQ * PASS_NV;
        for (int o = tid; o < TQ * PASS_NV; o += PASS_THREADS) {
            const int qq = o / PASS_NV, v = o - qq * PASS_NV;
            double s = 0.0;
            for (int f = 0; f < nper; f++) s += s_red[v][qq * nper + f];
            out[o] = s;
        }
    };

    for (int64_t u = u_begin; u < u_end; u++) {
        const int64_t ru = u / g.TC;
        const int tc = (int)(u - ru * g.TC);
        int c = cur_c;
        if (c < 0 || ru < g.cum(c) || (c < g.ncols - 1 && ru >= g.cum(c + 1))) c = g.col_of(ru);
        const int p = (int)(ru - g.cum(c));
        if (c != cur_c) {
            if (cur_c >= 0) flush_q(cur_c);
            cur_c = c;
            sq.zero();
            q = TQ * c + ql;
            load_jones(jones + (size_t)min(q, N - 1) * 4, Jq);
            gram(Jq, hq00, hq11, hq01);
        }
        if (p != cur_p) {
            cur_p = p;
            load_jones(jones + (size_t)p * 4, Jp);
            gram(Jp, hp00, hp11, hp01);
        }
        const bool valid = thread_used && q > p && q < N;
        const int t0 = tc * g.tlen, t1 = min(g.T, t0 + g.tlen);
        Side sp;
        sp.zero();
        double cost = 0.0;
        if (valid) {
            const int64_t b = bl_index(N, p, q);
            {
                // C = c*I2: model = c (J_p J_q^H); S = sum conj(c) E; s2 = sum |c|^2
                m22 P;
                mmh(Jp, Jq, P);
                cplx S[4] = {mk(0, 0), mk(0, 0), mk(0, 0), mk(0, 0)};
                double s2 = 0.0;
                for (int j = 0; j < g.nchunk; j++) {
                    const int f = g.nchunk > 1 ? tid + j * PASS_THREADS : tid - ql * F;
                    if (f >= F) break;
                    for (int t = t0; t < t1; t++) {
                        const size_t idx = ((size_t)t * g.B + b) * F + f;
                        m22 X;
                        load_m22_stream(x + idx * 4, X);
                        const cplx cc = ldg128_stream(coh + idx);
#pragma unroll
                        for (int i = 0; i < 4; i++) {
                            const cplx e = cfms(cc, P.a[i], X.a[i]);
                            cost = cabs2(e, cost);
                            S[i] = cfmaca(cc, e, S[i]);
                        }
                        s2 = cabs2(cc, s2);
                    }
                }
                // G_p += S J_q;  G_q += S^H J_p;  M_p += s2 J_q^H J_q;  M_q += s2 J_p^H J_p
                sp.G[0] = cfma(S[1], Jq.a[2], cmul(S[0], Jq.a[0]));
                sp.G[1] = cfma(S[1], Jq.a[3], cmul(S[0], Jq.a[1]));
                sp.G[2] = cfma(S[3], Jq.a[2], cmul(S[2], Jq.a[0]));
                sp.G[3] = cfma(S[3], Jq.a[3], cmul(S[2], Jq.a[1]));
                sq.G[0] = cfmaca(S[2], Jp.a[2], cfmaca(S[0], Jp.a[0], sq.G[0]));
                sq.G[1] = cfmaca(S[2], Jp.a[3], cfmaca(S[0], Jp.a[1], sq.G[1]));
                sq.G[2] = cfmaca(S[3], Jp.a[2], cfmaca(S[1], Jp.a[0], sq.G[2]));
                sq.G[3] = cfmaca(S[3], Jp.a[3], cfmaca(S[1], Jp.a[1], sq.G[3]));
                sp.M00 = s2 * hq00; sp.M11 = s2 * hq11; sp.M01 = mk(s2 * hq01.re, s2 * hq01.im);
                sq.M00 = fma(s2, hp00, sq.M00); sq.M11 = fma(s2, hp11, sq.M11);
                sq.M01 = mk(fma(s2, hp01.re, sq.M01.re), fma(s2, hp01.im, sq.M01.im));
            }
        }
        // p side: warp-shuffle reduction, one record per (unit, warp)
        double* pp = Ppart + ((size_t)u * PASS_WARPS + warp) * PASS_NV;
#pragma unroll
        for (int i = 0; i < PASS_NV; i++) {
            const double s = warp_sum(sp.get(i));
            if (lane == 0) pp[i] = s;
        }
        const double cs = warp_sum(cost);
        if (lane == 0) Pcost[(size_t)u * PASS_WARPS + warp] = cs;
    }
    if (cur_c >= 0) flush_q(cur_c);
}

// ---- fixed-order station reduction ------------------------------------------------------------------------------
// block s < N: station s;  block N: cost.
constexpr int RED_THREADS = 128;

__global__ void __launch_bounds__(RED_THREADS)
lm_reduce_kernel(PassGeom g, const double* __restrict__ Ppart, const double* __restrict__ Pcost,
                 const double* __restrict__ Qpart, double* __restrict__ cost, sagecal_c128* __restrict__ grad,
                 sagecal_c128* __restrict__ jtj) {
    __shared__ double s_red[PASS_NV][RED_THREADS];
    const int tid = threadIdx.x;
    const int s = blockIdx.x;
    double acc[PASS_NV];
#pragma unroll
    for (int i = 0; i < PASS_NV; i++) acc[i] = 0.0;

    if (s == g.N) {  // cost: sum of all Pcost entries
        const int64_t n = g.U * PASS_WARPS;
        for (int64_t i = tid; i < n; i += RED_THREADS) acc[0] += Pcost[i];
    } else {
        // p side: units (c, p=s, tc) of every column that has row s: q range must reach beyond s
        const int per_row = g.TC * PASS_WARPS;  // contiguous records per (column,row)
        const int cmin = (s + 1) / g.TQ;        // column holding q = s+1
        for (int c = cmin; c < g.ncols; c++) {
            if (g.qhi(c) - 1 <= s) continue;
            const double* base = Ppart + (size_t)(g.cum(c) + s) * per_row * PASS_NV;
            for (int e = tid; e < per_row; e += RED_THREADS) {
#pragma unroll
                for (int i = 0; i < PASS_NV; i++) acc[i] += base[(size_t)e * PASS_NV + i];
            }
        }
        // q side: one record per slot that touched column c = s / TQ
        const int c = s / g.TQ;
        const int64_t nrows_c = g.qhi(c) - 1;
        if (nrows_c > 0) {
            const int64_t ub = g.cum(c) * g.TC, ue = (g.cum(c) + nrows_c) * g.TC;
            const int i0 = g.slot_of(ub), i1 = g.slot_of(ue - 1);
            for (int i = i0 + tid; i <= i1; i += RED_THREADS) {
                const double* rec = Qpart + ((size_t)(i + c) * g.TQ + (s - g.TQ * c)) * PASS_NV;
#pragma unroll
                for (int v = 0; v < PASS_NV; v++) acc[v] += rec[v];
            }
        }
    }
#pragma unroll
    for (int i = 0; i < PASS_NV; i++) s_red[i][tid] = acc[i];
    __syncthreads();
    for (int o = RED_THREADS / 2; o > 0; o >>= 1) {
        if (tid < o) {
#pragma unroll
            for (int i = 0; i < PASS_NV; i++) s_red[i][tid] += s_red[i][tid + o];
        }
        __syncthreads();
    }
    if (tid == 0) {
        if (s == g.N) {
            *cost = s_red[0][0];
        } else {
            sagecal_c128* G = grad + (size_t)s * 4;
            sagecal_c128* M = jtj + (size_t)s * 4;
            for (int i = 0; i < 4; i++) { G[i].re = s_red[2 * i][0]; G[i].im = s_red[2 * i + 1][0]; }
            M[0].re = s_red[8][0];  M[0].im = 0.0;
            M[1].re = s_red[10][0]; M[1].im = s_red[11][0];
            M[2].re = s_red[10][0]; M[2].im = -s_red[11][0];
            M[3].re = s_red[9][0];  M[3].im = 0.0;
        }
    }
}

int enqueue_pass(const PassGeom& g, const PassWorkspace& w, const sagecal_c128* x, int coh_format,
                 const sagecal_c128* coh_k, const sagecal_c128* jones, double* cost, sagecal_c128* grad,
                 sagecal_c128* jtj, cudaStream_t st) {
    // 2x2 coherencies: the tensor-core form (lm_pass_mma.cu); the kernel below then serves the scalar form
    if (coh_format != SAGECAL_COH_SCALAR) return enqueue_pass_mma(g, w, x, coh_k, jones, cost, grad, jtj, st);
    {
        LaunchScope ls(KK_PASS, st);
        lm_pass_scalar_kernel<<<g.nslots, PASS_THREADS, 0, st>>>(g, x, coh_k, jones, w.Ppart, w.Pcost, w.Qpart);
        SGC_LAUNCH_CHECK();
    }
    {
        LaunchScope ls(KK_REDUCE, st);
        lm_reduce_kernel<<<g.N + 1, RED_THREADS, 0, st>>>(g, w.Ppart, w.Pcost, w.Qpart, cost, grad, jtj);
        SGC_LAUNCH_CHECK();
    }
    return SAGECAL_OK;
}

}  // namespace sgc

using namespace sgc;

extern "C" int sagecal_lm_cost_grad_jtj(int N, int T, int F, const sagecal_c128* x, int coh_format,
                                        const sagecal_c128* coh_k, const sagecal_c128* jones_k, double* cost,
                                        sagecal_c128* grad, sagecal_c128* jtj, void* workspace,
                                        size_t workspace_bytes, void* stream) {
    if (N < 2 || T < 1 || F < 1) return SAGECAL_EINVAL;
    if (coh_format != SAGECAL_COH_FULL && coh_format != SAGECAL_COH_SCALAR) return SAGECAL_EINVAL;
    if (!x || !coh_k || !jones_k || !cost || !grad || !jtj) return SAGECAL_EINVAL;
    if (!aligned(x, 32) || !aligned(coh_k, coh_format == SAGECAL_COH_SCALAR ? 16 : 32) || !aligned(jones_k, 16) ||
        !aligned(grad, 16) || !aligned(jtj, 16) || !aligned(cost, 8))
        return SAGECAL_EINVAL;
    const PassGeom g = make_pass_geom(N, T, F);
    if (!workspace || !aligned(workspace, 256) || workspace_bytes < pass_workspace_bytes(g)) return SAGECAL_EWORKSPACE;
    const PassWorkspace w = carve_pass_workspace(g, workspace);
    return enqueue_pass(g, w, x, coh_format, coh_k, jones_k, cost, grad, jtj, (cudaStream_t)stream);
}

// Host-side replay of the pass kernel's work decomposition, for CPU tests of the geometry (no device needed):
// cover[t*B + b] counts how many (slot, unit, thread) visits reach baseline b at time t (must be exactly 1);
// the return value is non-zero if the partial-sum bookkeeping the reduction kernel relies on is inconsistent.
// info[0..7] = {TQ, nchunk, ncols, TC, tlen, nslots, R, U}.
extern "C" int sagecal_debug_pass_cover(int N, int T, int F, int32_t* cover, int64_t* info) {
    if (N < 2 || T < 1 || F < 1 || !cover || !info) return SAGECAL_EINVAL;
    const PassGeom g = make_pass_geom(N, T, F);
    info[0] = g.TQ; info[1] = g.nchunk; info[2] = g.ncols; info[3] = g.TC;
    info[4] = g.tlen; info[5] = g.nslots; info[6] = g.R; info[7] = g.U;
    int bad = 0;
    const int nrec = g.nslots + g.ncols;
    int* rec_col = new int[nrec];
    for (int i = 0; i < nrec; i++) rec_col[i] = -1;
    if (g.slot_begin(0) != 0 || g.slot_begin(g.nslots) != g.U) bad |= 1;
    for (int slot = 0; slot < g.nslots; slot++) {
        if (g.slot_begin(slot + 1) <= g.slot_begin(slot)) bad |= 2;  // every slot owns at least one unit
        int cur_c = -1;
        for (int64_t u = g.slot_begin(slot); u < g.slot_begin(slot + 1); u++) {
            if (g.slot_of(u) != slot) bad |= 4;
            const int64_t ru = u / g.TC;
            const int tc = (int)(u - ru * g.TC);
            const int c = g.col_of(ru);
            const int p = (int)(ru - g.cum(c));
            if (p < 0 || p >= g.qhi(c) - 1) bad |= 8;
            if (c != cur_c) {
                if (c < cur_c) bad |= 16;
                if (rec_col[slot + c] != -1) bad |= 32;  // record index slot+column must be unique
                rec_col[slot + c] = c;
                cur_c = c;
            }
            const int t0 = tc * g.tlen, t1 = t0 + g.tlen < T ? t0 + g.tlen : T;
            for (int ql = 0; ql < g.TQ; ql++) {
                const int q = g.TQ * c + ql;
                if (q > p && q < N)
                    for (int t = t0; t < t1; t++) cover[(int64_t)t * g.B + bl_index(N, p, q)]++;
            }
        }
    }
    // the reduction's view: column c is touched by exactly the slots slot_of(first unit) .. slot_of(last unit)
    for (int c = 0; c < g.ncols; c++) {
        const int64_t nrows = g.qhi(c) - 1;
        int expect = 0;
        if (nrows > 0) {
            const int i0 = g.slot_of(g.cum(c) * g.TC), i1 = g.slot_of((g.cum(c) + nrows) * g.TC - 1);
            for (int i = i0; i <= i1; i++, expect++)
                if (rec_col[i + c] != c) bad |= 64;
        }
        int have = 0;
        for (int i = 0; i < nrec; i++) have += rec_col[i] == c;
        if (have != expect) bad |= 128;
    }
    delete[] rec_col;
    return bad;
}
