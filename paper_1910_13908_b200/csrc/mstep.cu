// One chunk of a compressed M-step as ONE cooperative kernel (formulas: compress.cuh): the initial
// evaluation at the centre Jones and n_trial Levenberg-Marquardt trial steps, each = cost / gradient / per-station
// J^H J from the per-baseline statistics (rows 8a-4, 8a-5 of SURVEY.md §8(a) re-associated), with the damping,
// accept/reject and 2x2 solves on the device and grid-wide barriers between the phases:
//
//   A  tiles   : CTA <- tile (PB row stations p x 32 column stations q), walked in steps of 2 rows.  The step's
//                statistics (2 x 32 records) are staged in shared memory with cp.async one step ahead of the
//                arithmetic; the tile's Jones (trial, centre, difference, Gram matrix) are staged once.
//                4 lanes share one baseline, lane a = 2i+j owns row a of dW / Sec, i.e. residual entry (i, j): it
//                needs only row i of J_p and row j of J_q.  Row-station sums: shuffles over the lanes, combined over
//                the 4 warps of a row in shared memory, one record per (column tile, row).  Column-station sums:
//                registers over the rows, combined over the 2 row groups in shared memory, one record per
//                (row block, column).  Cost: one sum per CTA.
//      -- grid barrier --
//   B  control : every warp adds the CTA costs and the stations' predicted reductions in the same fixed order
//                (identical in all CTAs), takes the accept/reject decision and updates mu, nu.  Warp <-> station:
//                adds the station's records (lanes over records, butterfly), commits or discards the trial, solves
//                dJ_p = G_p (M_p + mu I)^-1, writes the next trial Jones, its Gram matrix and predicted reduction.
//      -- grid barrier --
//
// No atomics in the sums, fixed summation order: bit-reproducible for a given grid.  The launch is cooperative, so
// all CTAs are co-resident; the grid barrier is an arrive counter in device memory (one red.release per CTA, relaxed
// polling, one acquire fence).  cooperative_groups' grid.sync() is faster in isolation (1.3 vs 1.5 us at 272 CTAs)
// but makes every warp invalidate its L1 (CCTL.IVALL), after which the loads of phase B took 17 us instead of 2 us
// here; all data that crosses CTAs is read with ld.cg / cp.async.cg (L2), so no L1 invalidation is needed.
// The statistics (400 B per baseline, 52 MB at N=512) stay L2-resident over the evaluations.
#include <math.h>
#include "compress.cuh"

namespace sgc {

struct MstepArgs {
    MGeom g;
    int lpb;                   // log2(PB)
    const double *Src, *Scc;
    double *Ppart, *Qpart, *cost_cta, *pred_st, *mm_st, *Htry;
    sagecal_c128 *G, *M, *J_try, *J0, *Jk;
    MstepCtl* ctl;
    unsigned* bar;
    int n_trial, init;
    double tau;
    double *cost_out, *trace_out;
};

// ---- small helpers ------------------------------------------------------------------------------------------------
__device__ __forceinline__ double wsum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ cplx ldcg_c(const sagecal_c128* p) {   // coherent at L2: data other CTAs write
    const double2 v = __ldcg(reinterpret_cast<const double2*>(p));
    return mk(v.x, v.y);
}
__device__ __forceinline__ void st_c(sagecal_c128* p, cplx v) { p->re = v.re; p->im = v.im; }
__device__ __forceinline__ cplx csub(cplx a, cplx b) { return mk(a.re - b.re, a.im - b.im); }
__device__ __forceinline__ cplx cadd(cplx a, cplx b) { return mk(a.re + b.re, a.im + b.im); }
__device__ __forceinline__ cplx lds_c(const double* p) {
    const double2 v = *reinterpret_cast<const double2*>(p);
    return mk(v.x, v.y);
}

// every lane of every warp gets the same sum: lane-strided partial sums (16 loads in flight), then a butterfly
__device__ __forceinline__ double strided_sum(const double* p, int n, int lane) {
    double v = 0.0;
    for (int base = 0; base < n; base += 512) {
        double t[16];
#pragma unroll
        for (int u = 0; u < 16; u++) {
            const int i = base + 32 * u + lane;
            t[u] = i < n ? __ldcg(p + i) : 0.0;
        }
#pragma unroll
        for (int u = 0; u < 16; u++) v += t[u];
    }
    return wsum(v);
}
__device__ __forceinline__ double strided_max(const double* p, int n, int lane) {
    double v = 0.0;
    for (int base = 0; base < n; base += 256) {
        double t[8];
#pragma unroll
        for (int u = 0; u < 8; u++) {
            const int i = base + 32 * u + lane;
            t[u] = i < n ? __ldcg(p + i) : 0.0;
        }
#pragma unroll
        for (int u = 0; u < 8; u++) v = fmax(v, t[u]);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

// ---- grid barrier: arrive counter, generation gen = 1, 2, ... (the counter is zeroed before every launch) ----------
__device__ __forceinline__ void grid_barrier(unsigned* bar, unsigned gen) {
    __syncthreads();
    if (threadIdx.x == 0) {
        asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(bar) : "memory");
        unsigned v;
        do {
            asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(bar) : "memory");
        } while (v < gridDim.x * gen);
        asm volatile("fence.acq_rel.gpu;" ::: "memory");
    }
    __syncthreads();
}

// ---- shared-memory staging ----------------------------------------------------------------------------------------
__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async8(void* smem, const void* gmem) {
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(s), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N_>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N_) : "memory"); }

// record strides (bytes); in shared memory the Scc record is padded by 16 B so that the 8 baselines of a warp fall
// into different banks.  Every warp stages its own rows (8 baselines each), double-buffered.
template <bool SCALAR> struct Stage {
    static constexpr int SRC_B = (SCALAR ? NSRC_SCALAR : NSRC_FULL) * 8;          // 80 / 272
    static constexpr int SCC_G = (SCALAR ? NSCC_SCALAR : NSCC_FULL) * 8;          // 8 / 128 in global memory
    static constexpr int SCC_S = SCALAR ? 8 : 144;                                // in shared memory
    static constexpr int SRC_W = 8 * SRC_B;                                       // the 8 Src records of a warp's row
    static constexpr int WROW_B = 8 * (SRC_B + SCC_S);                            // one row of one warp
    static constexpr int ALL_B = MS_WARPS * 2 * WROW_B;
};
constexpr int JST = 28;     // doubles per staged station: J_try (8), J0 (8), D = J_try - J0 (8), H = J_try^H J_try (4)

template <bool SCALAR>
constexpr size_t mstep_smem_bytes() {
    return (size_t)Stage<SCALAR>::ALL_B +
           sizeof(double) * ((MS_PB_MAX + MS_TQ) * JST + MS_PB_MAX * 4 * MS_NV + 2 * MS_TQ * MS_NV + MS_WARPS);
}

struct Herm { double h00, h11; cplx h01; };

// ---- one lane's share of one baseline -----------------------------------------------------------------------------
// lane a = 2i+j.  prow / pcol: the staged records (JST doubles: J_try, J0, D, H) of the row station p and the column
// station q; the lane needs row i of J_p, D_p and row j of J_q, J0_q, D_q, read from shared memory where they are
// used so that few values are live at a time.  src / scc: this baseline's staged statistics.
// gp += its part of G_p row i;  gqc = its part of G_q row j;  mp / mq: a=0 (M_p00, M_p11), a=1 M_p01, a=2 (M_q00, M_q11),
// a=3 M_q01.
__device__ __forceinline__ Herm lds_herm(const double* rec) {
    Herm h; h.h00 = rec[24]; h.h11 = rec[25]; h.h01 = mk(rec[26], rec[27]);
    return h;
}
template <bool SCALAR>
__device__ __forceinline__ void lane_task(const double* src, const double* scc, int a, const double* prow,
                                          const double* pcol, cplx* gp, cplx* gqc, double* mp, double* mq, double& cost) {
    const int i = a >> 1, j = a & 1;
    const double* jp_ = prow + 4 * i;            // row i of J_p (trial)
    const double* dp_ = prow + 16 + 4 * i;       // row i of D_p
    const double* jq_ = pcol + 4 * j;            // row j of J_q (trial)
    const double* jq0_ = pcol + 8 + 4 * j;       // row j of J0_q
    const double* dq_ = pcol + 16 + 4 * j;       // row j of D_q
    if (SCALAR) {
        const double s2 = scc[0];
        const cplx sr = lds_c(src + 2 * a);
        const cplx jp[2] = {lds_c(jp_), lds_c(jp_ + 2)};
        // dP[(i,j)] = sum_k D_p[i,k] conj(J0_q[j,k]) + J_p[i,k] conj(D_q[j,k])
        cplx dP = cmulc(lds_c(dp_), lds_c(jq0_));
        dP = cfmac(lds_c(dp_ + 2), lds_c(jq0_ + 2), dP);
        dP = cfmac(jp[0], lds_c(dq_), dP);
        dP = cfmac(jp[1], lds_c(dq_ + 2), dP);
        const cplx se = mk(fma(-s2, dP.re, sr.re), fma(-s2, dP.im, sr.im));
        const double acc = fma(dP.re, sr.re + se.re, dP.im * (sr.im + se.im));
        cost += (a == 0 ? src[NSRC_SCALAR - 2] : 0.0) - acc;
        gp[0] = cfma(se, lds_c(jq_), gp[0]);      // G_p[i,k] += Se[(i,j)] J_q[j,k]
        gp[1] = cfma(se, lds_c(jq_ + 2), gp[1]);
        gqc[0] = cmulc(jp[0], se);                // G_q[j,l] += conj(Se[(i,j)]) J_p[i,l]
        gqc[1] = cmulc(jp[1], se);
        const Herm h = lds_herm(a < 2 ? pcol : prow);
        if (a == 0) { mp[0] = fma(s2, h.h00, mp[0]); mp[1] = fma(s2, h.h11, mp[1]); }
        else if (a == 1) { mp[0] = fma(s2, h.h01.re, mp[0]); mp[1] = fma(s2, h.h01.im, mp[1]); }
        else if (a == 2) { mq[0] = fma(s2, h.h00, mq[0]); mq[1] = fma(s2, h.h11, mq[1]); }
        else { mq[0] = fma(s2, h.h01.re, mq[0]); mq[1] = fma(s2, h.h01.im, mq[1]); }
        return;
    }
    // row a of dW: dW[(k,l)] = D_p[i,k] conj(J0_q[j,l]) + J_p[i,k] conj(D_q[j,l])
    cplx dW[4];
    {
        const cplx dp[2] = {lds_c(dp_), lds_c(dp_ + 2)}, jq0[2] = {lds_c(jq0_), lds_c(jq0_ + 2)};
        const cplx jp[2] = {lds_c(jp_), lds_c(jp_ + 2)}, dq[2] = {lds_c(dq_), lds_c(dq_ + 2)};
#pragma unroll
        for (int c = 0; c < 4; c++) dW[c] = cfmac(jp[c >> 1], dq[c & 1], cmulc(dp[c >> 1], jq0[c & 1]));
    }
    // Hermitian Scc: S[0][0], S[1][1], S[2][2], S[3][3], then (0,1) (0,2) (0,3) (1,2) (1,3) (2,3)
    cplx S[4][4];
    {
        const double2 d0 = *reinterpret_cast<const double2*>(scc), d1 = *reinterpret_cast<const double2*>(scc + 2);
        S[0][0] = mk(d0.x, 0.0); S[1][1] = mk(d0.y, 0.0); S[2][2] = mk(d1.x, 0.0); S[3][3] = mk(d1.y, 0.0);
        S[0][1] = lds_c(scc + 4); S[0][2] = lds_c(scc + 6); S[0][3] = lds_c(scc + 8);
        S[1][2] = lds_c(scc + 10); S[1][3] = lds_c(scc + 12); S[2][3] = lds_c(scc + 14);
    }
#pragma unroll
    for (int x = 0; x < 4; x++) {
#pragma unroll
        for (int y = x + 1; y < 4; y++) S[y][x] = mk(S[x][y].re, -S[x][y].im);
    }
    // row a of Src (64 B), Sec = Src - dW Scc, cost
    const double* rp = src + 8 * a;
    cplx sec[4];
    double acc = 0.0;
#pragma unroll
    for (int c = 0; c < 4; c++) {
        const cplx sv = lds_c(rp + 2 * c);
        cplx t = sv;
#pragma unroll
        for (int d = 0; d < 4; d++) t = cfms(dW[d], S[d][c], t);
        sec[c] = t;
        acc = fma(dW[c].re, sv.re + t.re, fma(dW[c].im, sv.im + t.im, acc));
    }
    cost += (a == 0 ? src[NSRC_FULL - 2] : 0.0) - acc;
    // G_p[i,k] += sum_l J_q[j,l] Sec[(i,j),(k,l)];   G_q[j,l] += sum_k J_p[i,k] conj(Sec[(i,j),(k,l)])
    {
        const cplx jq[2] = {lds_c(jq_), lds_c(jq_ + 2)}, jp[2] = {lds_c(jp_), lds_c(jp_ + 2)};
        gp[0] = cfma(jq[1], sec[1], cfma(jq[0], sec[0], gp[0]));
        gp[1] = cfma(jq[1], sec[3], cfma(jq[0], sec[2], gp[1]));
        gqc[0] = cfmac(jp[1], sec[2], cmulc(jp[0], sec[0]));
        gqc[1] = cfmac(jp[1], sec[3], cmulc(jp[0], sec[1]));
    }
    const Herm h = lds_herm(a < 2 ? pcol : prow);     // Hq for the row station's M, Hp for the column station's
    if (a == 0) {          // M_p[k,k] = sum_{l,l'} Hq[l,l'] S[(k,l)][(k,l')]
        mp[0] += fma(h.h00, S[0][0].re, fma(h.h11, S[1][1].re, 2.0 * fma(h.h01.re, S[0][1].re, -h.h01.im * S[0][1].im)));
        mp[1] += fma(h.h00, S[2][2].re, fma(h.h11, S[3][3].re, 2.0 * fma(h.h01.re, S[2][3].re, -h.h01.im * S[2][3].im)));
    } else if (a == 1) {   // M_p[0,1] = Hq00 S[0][2] + Hq01 S[0][3] + conj(Hq01) S[1][2] + Hq11 S[1][3]
        cplx m = mk(h.h00 * S[0][2].re, h.h00 * S[0][2].im);
        m = cfma(h.h01, S[0][3], m);
        m = cfmaca(h.h01, S[1][2], m);
        mp[0] += fma(h.h11, S[1][3].re, m.re);
        mp[1] += fma(h.h11, S[1][3].im, m.im);
    } else if (a == 2) {   // M_q[l,l] = sum_{k,k'} Hp[k,k'] conj(S[(k,l)][(k',l)])
        mq[0] += fma(h.h00, S[0][0].re, fma(h.h11, S[2][2].re, 2.0 * fma(h.h01.re, S[0][2].re, h.h01.im * S[0][2].im)));
        mq[1] += fma(h.h00, S[1][1].re, fma(h.h11, S[3][3].re, 2.0 * fma(h.h01.re, S[1][3].re, h.h01.im * S[1][3].im)));
    } else {               // M_q[0,1] = Hp00 conj(S[0][1]) + Hp01 conj(S[0][3]) + conj(Hp01) S[1][2] + Hp11 conj(S[2][3])
        cplx m = mk(h.h00 * S[0][1].re, -h.h00 * S[0][1].im);
        m = cfmac(h.h01, S[0][3], m);
        m = cfmaca(h.h01, S[1][2], m);
        mq[0] += fma(h.h11, S[2][3].re, m.re);
        mq[1] += fma(-h.h11, S[2][3].im, m.im);
    }
}

// ---- phase A ------------------------------------------------------------------------------------------------------
struct Smem {
    unsigned char* stage;              // [MS_WARPS][2][WROW_B]
    double* jst;                       // [(MS_PB_MAX + MS_TQ)][JST]: the tile's rows, then its columns
    double (*s_p)[4][MS_NV];           // [MS_PB_MAX][4 column groups][12]
    double (*s_q)[MS_TQ][MS_NV];       // [2 row groups][32][12]
    double* s_cost;                    // [MS_WARPS]
};
template <bool SCALAR>
__device__ __forceinline__ Smem carve_smem(unsigned char* base) {
    Smem s;
    s.stage = base;
    double* d = reinterpret_cast<double*>(base + Stage<SCALAR>::ALL_B);
    s.jst = d; d += (MS_PB_MAX + MS_TQ) * JST;
    s.s_p = reinterpret_cast<double (*)[4][MS_NV]>(d); d += MS_PB_MAX * 4 * MS_NV;
    s.s_q = reinterpret_cast<double (*)[MS_TQ][MS_NV]>(d); d += 2 * MS_TQ * MS_NV;
    s.s_cost = d;
    return s;
}

// cp.async the statistics of row r of tile (qt, pb), columns 8*sq .. 8*sq+7, into the warp's buffer `buf`
// (slot = column within the warp's 8); the lanes of the warp share the 16-byte chunks
template <bool SCALAR>
__device__ __forceinline__ void issue_row(const MstepArgs& A, unsigned char* buf, int qt, int pb, int sq, int r, int lane) {
    using St = Stage<SCALAR>;
    const int N = A.g.N;
    const int p = (pb << A.lpb) + r;
    if (p >= N - 1) return;
    const int qw0 = MS_TQ * qt + 8 * sq;
    const int qlo = max(qw0, p + 1), qhi = min(qw0 + 8, N), cnt = qhi - qlo;
    if (cnt <= 0) return;
    const int64_t b0 = bl_index(N, p, qlo);
    {
        const unsigned char* g = reinterpret_cast<const unsigned char*>(A.Src) + (size_t)b0 * St::SRC_B;
        unsigned char* d = buf + (qlo - qw0) * St::SRC_B;
        const int nchunk = cnt * (St::SRC_B / 16);
        for (int c = lane; c < nchunk; c += 32) cp_async16(d + 16 * c, g + 16 * c);
    }
    {
        const unsigned char* g = reinterpret_cast<const unsigned char*>(A.Scc) + (size_t)b0 * St::SCC_G;
        unsigned char* d = buf + St::SRC_W + (qlo - qw0) * St::SCC_S;
        if (SCALAR) {
            if (lane < cnt) cp_async8(d + 8 * lane, g + 8 * lane);
        } else {
            for (int c = lane; c < cnt * 8; c += 32) cp_async16(d + (c >> 3) * St::SCC_S + (c & 7) * 16, g + 16 * c);
        }
    }
}

template <bool SCALAR>
__device__ __forceinline__ void phase_tiles(const MstepArgs& A, const Smem& sm) {
    using St = Stage<SCALAR>;
    const MGeom& g = A.g;
    const int N = g.N, PB = g.PB, lpb = A.lpb;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int sq = warp & 3, rg = warp >> 2;
    const int qi = lane >> 2, a = lane & 3;
    const int ql = 8 * sq + qi;
    const int nsteps = PB >> 1;
    double cost = 0.0;
    for (int tile = blockIdx.x; tile < g.ntiles; tile += gridDim.x) {
        int qt = 0, pb = tile;
        for (;;) {
            const int nl = (g.qmax(qt) + PB - 1) >> lpb;
            if (pb < nl) break;
            pb -= nl; qt++;
        }
        unsigned char* wbuf = sm.stage + warp * 2 * St::WROW_B;
        issue_row<SCALAR>(A, wbuf, qt, pb, sq, rg, lane);
        cp_async_commit();
        // the tile's Jones: rows then columns; per station J_try, J0, D = J_try - J0, H
        for (int o = tid; o < (PB + MS_TQ) * 5; o += MS_THREADS) {
            const int st = o / 5, x = o - st * 5;
            const int s = st < PB ? min((pb << lpb) + st, N - 1) : min(MS_TQ * qt + (st - PB), N - 1);
            double* rec = sm.jst + (st < PB ? st : MS_PB_MAX + (st - PB)) * JST;
            if (x < 4) {
                const cplx jt = ldcg_c(A.J_try + 4 * s + x), j0 = ldcg_c(A.J0 + 4 * s + x);
                rec[2 * x] = jt.re; rec[2 * x + 1] = jt.im;
                rec[8 + 2 * x] = j0.re; rec[9 + 2 * x] = j0.im;
                rec[16 + 2 * x] = jt.re - j0.re; rec[17 + 2 * x] = jt.im - j0.im;
            } else {
                const double2 h0 = __ldcg(reinterpret_cast<const double2*>(A.Htry + 4 * s));
                const double2 h1 = __ldcg(reinterpret_cast<const double2*>(A.Htry + 4 * s + 2));
                rec[24] = h0.x; rec[25] = h0.y; rec[26] = h1.x; rec[27] = h1.y;
            }
        }
        const int q = MS_TQ * qt + ql;
        const double* pcol = sm.jst + (MS_PB_MAX + ql) * JST;
        cplx gq[2] = {mk(0.0, 0.0), mk(0.0, 0.0)};
        double mq[2] = {0.0, 0.0};
        __syncthreads();                                            // the staged Jones are visible
        for (int step = 0; step < nsteps; step++) {
            const int r = 2 * step + rg, p = (pb << lpb) + r;
            if (step + 1 < nsteps) issue_row<SCALAR>(A, wbuf + ((step + 1) & 1) * St::WROW_B, qt, pb, sq, r + 2, lane);
            cp_async_commit();
            cp_async_wait<1>();
            __syncwarp();
            if (p < N - 1) {                                        // warp-uniform
                cplx gp[2] = {mk(0.0, 0.0), mk(0.0, 0.0)}, gqc[2] = {mk(0.0, 0.0), mk(0.0, 0.0)};
                double mp[2] = {0.0, 0.0};
                if (q < N && q > p) {
                    const unsigned char* row = wbuf + (step & 1) * St::WROW_B;
                    lane_task<SCALAR>(reinterpret_cast<const double*>(row + qi * St::SRC_B),
                                      reinterpret_cast<const double*>(row + St::SRC_W + qi * St::SCC_S), a,
                                      sm.jst + r * JST, pcol, gp, gqc, mp, mq, cost);
                }
                // row station: G_p row i over j (xor 1) and the 8 columns (xor 4, 8, 16); M slots over the columns
                double v[6] = {gp[0].re, gp[0].im, gp[1].re, gp[1].im, mp[0], mp[1]};
#pragma unroll
                for (int x = 0; x < 4; x++) v[x] += __shfl_xor_sync(0xffffffffu, v[x], 1);
#pragma unroll
                for (int o = 4; o <= 16; o <<= 1) {
#pragma unroll
                    for (int x = 0; x < 6; x++) v[x] += __shfl_xor_sync(0xffffffffu, v[x], o);
                }
                if (qi == 0) {
                    double* out = sm.s_p[r][sq];
                    if (a == 0) { out[0] = v[0]; out[1] = v[1]; out[2] = v[2]; out[3] = v[3]; out[8] = v[4]; out[9] = v[5]; }
                    else if (a == 1) { out[10] = v[4]; out[11] = v[5]; }
                    else if (a == 2) { out[4] = v[0]; out[5] = v[1]; out[6] = v[2]; out[7] = v[3]; }
                }
                // column station: G_q row j over i (xor 2), accumulated over the rows
#pragma unroll
                for (int l = 0; l < 2; l++) {
                    gq[l].re += gqc[l].re + __shfl_xor_sync(0xffffffffu, gqc[l].re, 2);
                    gq[l].im += gqc[l].im + __shfl_xor_sync(0xffffffffu, gqc[l].im, 2);
                }
            }
            __syncwarp();                                           // the buffer is refilled two rows later
        }
        {
            double* out = sm.s_q[rg][ql];
            if (a == 0) { out[0] = gq[0].re; out[1] = gq[0].im; out[2] = gq[1].re; out[3] = gq[1].im; }
            else if (a == 1) { out[4] = gq[0].re; out[5] = gq[0].im; out[6] = gq[1].re; out[7] = gq[1].im; }
            else if (a == 2) { out[8] = mq[0]; out[9] = mq[1]; }
            else { out[10] = mq[0]; out[11] = mq[1]; }
        }
        __syncthreads();
        for (int o = tid; o < PB * MS_NV; o += MS_THREADS) {
            const int r = o / MS_NV, x = o - r * MS_NV, p = (pb << lpb) + r;
            if (p < N - 1)
                A.Ppart[((size_t)qt * N + p) * MS_NV + x] = ((sm.s_p[r][0][x] + sm.s_p[r][1][x]) + sm.s_p[r][2][x]) + sm.s_p[r][3][x];
        }
        for (int o = tid; o < MS_TQ * MS_NV; o += MS_THREADS) {
            const int c = o / MS_NV, x = o - c * MS_NV, qq = MS_TQ * qt + c;
            if (qq < N) A.Qpart[((size_t)pb * N + qq) * MS_NV + x] = sm.s_q[0][c][x] + sm.s_q[1][c][x];
        }
        __syncthreads();
    }
    cp_async_wait<0>();
    cost = wsum(cost);
    if (lane == 0) sm.s_cost[warp] = cost;
    __syncthreads();
    if (tid == 0) {
        double c = sm.s_cost[0];
#pragma unroll
        for (int w = 1; w < MS_WARPS; w++) c += sm.s_cost[w];
        A.cost_cta[blockIdx.x] = c;
    }
}

// ---- phase B helpers ----------------------------------------------------------------------------------------------
struct StAcc { cplx g[4]; cplx m[4]; };

// adds station s's records: lanes over records, butterfly; every lane returns the sums
__device__ __forceinline__ StAcc station_reduce(const MstepArgs& A, int s, int lane) {
    const MGeom& g = A.g;
    const int N = g.N;
    double acc[MS_NV];
#pragma unroll
    for (int x = 0; x < MS_NV; x++) acc[x] = 0.0;
    if (s <= N - 2) {
        for (int qt = (s + 1) / MS_TQ + lane; qt < g.nqt; qt += 32) {
            const double2* rec = reinterpret_cast<const double2*>(A.Ppart + ((size_t)qt * N + s) * MS_NV);
#pragma unroll
            for (int x = 0; x < MS_NV / 2; x++) { const double2 t = __ldcg(rec + x); acc[2 * x] += t.x; acc[2 * x + 1] += t.y; }
        }
    }
    if (s >= 1) {
        const int nl = (g.qmax(s / MS_TQ) + g.PB - 1) >> A.lpb;
        for (int pb = lane; pb < nl; pb += 32) {
            const double2* rec = reinterpret_cast<const double2*>(A.Qpart + ((size_t)pb * N + s) * MS_NV);
#pragma unroll
            for (int x = 0; x < MS_NV / 2; x++) { const double2 t = __ldcg(rec + x); acc[2 * x] += t.x; acc[2 * x + 1] += t.y; }
        }
    }
#pragma unroll
    for (int x = 0; x < MS_NV; x++) acc[x] = wsum(acc[x]);
    StAcc r;
#pragma unroll
    for (int x = 0; x < 4; x++) r.g[x] = mk(acc[2 * x], acc[2 * x + 1]);
    r.m[0] = mk(acc[8], 0.0); r.m[1] = mk(acc[10], acc[11]); r.m[2] = mk(acc[10], -acc[11]); r.m[3] = mk(acc[9], 0.0);
    return r;
}

// dJ = G (M + mu I)^-1, J_try = J + dJ; writes the trial Jones, its Gram matrix and this station's predicted
// reduction Re tr(G^H dJ) + mu ||dJ||^2
__device__ __forceinline__ void trial_step(const MstepArgs& A, int s, int lane, const cplx* g, const cplx* m,
                                           const cplx* jj, double mu, double* pred_out) {
    const double a = m[0].re + mu, d = m[3].re + mu;
    const cplx b = m[1];
    const double det = a * d - (b.re * b.re + b.im * b.im);
    const cplx inv[4] = {mk(d / det, 0.0), mk(-b.re / det, -b.im / det), mk(-b.re / det, b.im / det), mk(a / det, 0.0)};
    cplx dj[4], jt[4];
    dj[0] = cfma(g[1], inv[2], cmul(g[0], inv[0]));
    dj[1] = cfma(g[1], inv[3], cmul(g[0], inv[1]));
    dj[2] = cfma(g[3], inv[2], cmul(g[2], inv[0]));
    dj[3] = cfma(g[3], inv[3], cmul(g[2], inv[1]));
    double pred = 0.0;
#pragma unroll
    for (int x = 0; x < 4; x++) {
        jt[x] = cadd(jj[x], dj[x]);
        pred += g[x].re * dj[x].re + g[x].im * dj[x].im;
        pred += mu * (dj[x].re * dj[x].re + dj[x].im * dj[x].im);
    }
    if (lane == 0) {
#pragma unroll
        for (int x = 0; x < 4; x++) st_c(A.J_try + 4 * s + x, jt[x]);
        A.Htry[4 * s] = cabs2(jt[2], cabs2(jt[0], 0.0));          // H = J_try^H J_try
        A.Htry[4 * s + 1] = cabs2(jt[3], cabs2(jt[1], 0.0));
        const cplx h01 = cfmaca(jt[2], jt[3], cfmaca(jt[0], jt[1], mk(0.0, 0.0)));
        A.Htry[4 * s + 2] = h01.re;
        A.Htry[4 * s + 3] = h01.im;
        pred_out[s] = pred;
    }
}

template <bool SCALAR>
__global__ void __launch_bounds__(MS_THREADS, 2)
mstep_kernel(const MstepArgs A) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const Smem sm = carve_smem<SCALAR>(smem_raw);
    const int N = A.g.N;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int gw = blockIdx.x * MS_WARPS + warp, nw = gridDim.x * MS_WARPS;
    unsigned gen = 0;

    // LM state, identical in every thread of the grid
    double phi = 0.0, mu = A.init ? 0.0 : A.ctl->mu, nu = A.init ? 2.0 : A.ctl->nu;

    // prologue: centre and first "trial" = the current Jones of the cluster
    for (int s = gw; s < N; s += nw) {
        cplx jj[4];
#pragma unroll
        for (int x = 0; x < 4; x++) jj[x] = ldcg_c(A.Jk + 4 * s + x);
        if (lane == 0) {
#pragma unroll
            for (int x = 0; x < 4; x++) { st_c(A.J0 + 4 * s + x, jj[x]); st_c(A.J_try + 4 * s + x, jj[x]); }
            A.Htry[4 * s] = cabs2(jj[2], cabs2(jj[0], 0.0));
            A.Htry[4 * s + 1] = cabs2(jj[3], cabs2(jj[1], 0.0));
            const cplx h01 = cfmaca(jj[2], jj[3], cfmaca(jj[0], jj[1], mk(0.0, 0.0)));
            A.Htry[4 * s + 2] = h01.re;
            A.Htry[4 * s + 3] = h01.im;
        }
    }
    grid_barrier(A.bar, ++gen);

    for (int e = 0; e <= A.n_trial; e++) {
        phase_tiles<SCALAR>(A, sm);
        grid_barrier(A.bar, ++gen);

        const bool last = e == A.n_trial;
        if (e == 0 && A.init) {
            // (phi, G, M) at the centre are the accepted state; mu = tau * max_p max(M_p00, M_p11)
            for (int s = gw; s < N; s += nw) {
                const StAcc r = station_reduce(A, s, lane);
                if (lane == 0) {
#pragma unroll
                    for (int x = 0; x < 4; x++) { st_c(A.G + 4 * s + x, r.g[x]); st_c(A.M + 4 * s + x, r.m[x]); }
                    A.mm_st[s] = fmax(r.m[0].re, r.m[3].re);
                }
            }
            phi = strided_sum(A.cost_cta, (int)gridDim.x, lane);
            grid_barrier(A.bar, ++gen);
            mu = A.tau * strided_max(A.mm_st, N, lane);
            nu = 2.0;
            if (!(mu >= 1e-300)) mu = 1e-300;
            if (mu > 1e300) mu = 1e300;
            if (!last) {
                for (int s = gw; s < N; s += nw) {
                    cplx g4[4], m4[4], jj[4];
#pragma unroll
                    for (int x = 0; x < 4; x++) { g4[x] = ldcg_c(A.G + 4 * s + x); m4[x] = ldcg_c(A.M + 4 * s + x); jj[x] = ldcg_c(A.Jk + 4 * s + x); }
                    trial_step(A, s, lane, g4, m4, jj, mu, A.pred_st + (size_t)(e & 1) * N);
                }
            }
        } else {
            // this warp's first station: its loads are issued before the control sums so that both are in flight.
            // The accepted (G, M, J) and the trial J of a station are 16 complex numbers: lane x & 15 holds one.
            const int s0 = gw;
            const int which = lane & 15;
            auto old_elem = [&](int s) {
                const sagecal_c128* src = which < 4 ? A.G : which < 8 ? A.M : which < 12 ? A.Jk : A.J_try;
                return ldcg_c(src + 4 * s + (which & 3));
            };
            cplx mine = mk(0.0, 0.0);
            StAcc r0;
            if (s0 < N) {
                mine = old_elem(s0);
                r0 = station_reduce(A, s0, lane);
            }
            const double fresh = strided_sum(A.cost_cta, (int)gridDim.x, lane);
            bool accept = false;
            if (e == 0) {
                phi = fresh;                  // re-centre: fresh (phi, G, M) at the accepted Jones, mu and nu continue
            } else {
                // written by the stations' owners in the previous evaluation; this evaluation's go to the other half
                const double pred = strided_sum(A.pred_st + (size_t)((e - 1) & 1) * N, N, lane);
                const double rho = (phi - fresh) / pred;
                accept = isfinite(fresh) && isfinite(pred) && isfinite(rho) && pred > 0.0 && rho > 0.0;
                if (accept) {
                    phi = fresh;
                    const double t = 2.0 * rho - 1.0;
                    mu *= fmax(1.0 / 3.0, 1.0 - t * t * t);
                    nu = 2.0;
                } else {
                    mu *= nu;
                    nu *= 2.0;
                }
            }
            if (!(mu >= 1e-300)) mu = 1e-300;
            if (mu > 1e300) mu = 1e300;
            if (nu > 0x1p60) nu = 0x1p60;
            const bool take = accept || e == 0;
            for (int s = s0; s < N; s += nw) {
                StAcc r;
                if (s == s0) {
                    r = r0;
                } else {
                    mine = old_elem(s);
                    r = station_reduce(A, s, lane);
                }
                cplx g4[4], m4[4], jj[4];
#pragma unroll
                for (int x = 0; x < 4; x++) {
                    const int jsrc = accept ? 12 + x : 8 + x;
                    const cplx go = mk(__shfl_sync(0xffffffffu, mine.re, x), __shfl_sync(0xffffffffu, mine.im, x));
                    const cplx mo = mk(__shfl_sync(0xffffffffu, mine.re, 4 + x), __shfl_sync(0xffffffffu, mine.im, 4 + x));
                    jj[x] = mk(__shfl_sync(0xffffffffu, mine.re, jsrc), __shfl_sync(0xffffffffu, mine.im, jsrc));
                    g4[x] = take ? r.g[x] : go;
                    m4[x] = take ? r.m[x] : mo;
                }
                if (take && lane == 0) {
#pragma unroll
                    for (int x = 0; x < 4; x++) {
                        st_c(A.G + 4 * s + x, g4[x]); st_c(A.M + 4 * s + x, m4[x]);
                        if (accept) st_c(A.Jk + 4 * s + x, jj[x]);
                    }
                }
                if (!last) trial_step(A, s, lane, g4, m4, jj, mu, A.pred_st + (size_t)(e & 1) * N);
            }
        }
        if (!last) grid_barrier(A.bar, ++gen);
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        A.ctl->phi = phi; A.ctl->mu = mu; A.ctl->nu = nu;
        if (A.cost_out) *A.cost_out = phi;
        if (A.trace_out) *A.trace_out = phi;
    }
}

// ---- host side ----------------------------------------------------------------------------------------------------
// Rows per tile: the largest of 16, 8, 4, 2 that still gives about one tile per CTA slot of a B200 (148 SMs x 2);
// device independent, so the workspace can be sized without a device.
static int choose_pb(int N) {
    for (int PB = MS_PB_MAX; PB > 2; PB >>= 1)
        if (make_mgeom(N, PB).ntiles >= 252) return PB;
    return 2;
}
static int ilog2(int x) { int l = 0; while ((1 << l) < x) l++; return l; }

size_t compress_workspace_bytes(int N, int K, bool scalar) {
    const MGeom g = make_mgeom(N, choose_pb(N));
    size_t n = 0;
    n += round_up(sizeof(double) * (size_t)(K > 0 ? K : 1) * nscc(scalar) * g.B, 256);
    n += round_up(sizeof(double) * (size_t)nsrc(scalar) * g.B, 256);
    n += round_up(sizeof(double) * (size_t)g.nqt * N * MS_NV, 256);
    n += round_up(sizeof(double) * (size_t)g.npb * N * MS_NV, 256);
    n += round_up(sizeof(double) * MS_MAX_GRID, 256);
    n += round_up(sizeof(double) * 2 * (size_t)N, 256) + round_up(sizeof(double) * (size_t)N, 256);
    n += round_up(sizeof(double) * 4 * (size_t)N, 256);
    n += 3 * round_up((size_t)N * 64, 256);
    n += 256 + 256;
    n += round_up((size_t)2 * N * 64, 256);
    n += round_up(sizeof(double) * (size_t)GRP * nsrc(scalar) * g.B, 256);
    n += round_up(sizeof(double) * (size_t)ngroups(K > 0 ? K : 1) * GRP_PAIRS * nxg(scalar) * g.B, 256);
    n += round_up((size_t)2 * GRP * N * 64, 256);
    return n;
}

CompressWorkspace carve_compress(int N, int K, bool scalar, void* ws) {
    const MGeom g = make_mgeom(N, choose_pb(N));
    CompressWorkspace w;
    char* p = (char*)ws;
    auto take = [&](size_t n) { char* o = p; p += round_up(n, 256); return o; };
    w.Scc = (double*)take(sizeof(double) * (size_t)(K > 0 ? K : 1) * nscc(scalar) * g.B);
    w.Src = (double*)take(sizeof(double) * (size_t)nsrc(scalar) * g.B);
    w.Ppart = (double*)take(sizeof(double) * (size_t)g.nqt * N * MS_NV);
    w.Qpart = (double*)take(sizeof(double) * (size_t)g.npb * N * MS_NV);
    w.cost_cta = (double*)take(sizeof(double) * MS_MAX_GRID);
    w.pred_st = (double*)take(sizeof(double) * 2 * (size_t)N);
    w.mm_st = (double*)take(sizeof(double) * (size_t)N);
    w.Htry = (double*)take(sizeof(double) * 4 * (size_t)N);
    w.G = (sagecal_c128*)take((size_t)N * 64);
    w.M = (sagecal_c128*)take((size_t)N * 64);
    w.J_try = (sagecal_c128*)take((size_t)N * 64);
    w.ctl = (MstepCtl*)take(256);
    w.bar = (unsigned*)take(256);
    w.J0 = (sagecal_c128*)take((size_t)2 * N * 64);
    w.SrcG = (double*)take(sizeof(double) * (size_t)GRP * nsrc(scalar) * g.B);
    w.Xg = (double*)take(sizeof(double) * (size_t)ngroups(K > 0 ? K : 1) * GRP_PAIRS * nxg(scalar) * g.B);
    w.J0G = (sagecal_c128*)take((size_t)2 * GRP * N * 64);
    return w;
}

template <bool SCALAR>
static int max_coresident(int* out) {
    static int cached = 0;
    if (!cached) {
        int occ = 0;
        const size_t smem = mstep_smem_bytes<SCALAR>();
        SGC_CUDA(cudaFuncSetAttribute(mstep_kernel<SCALAR>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        SGC_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, mstep_kernel<SCALAR>, MS_THREADS, smem));
        if (occ < 1) return cuda_fail(cudaErrorLaunchOutOfResources);
        cached = occ * num_sms();
    }
    *out = cached;
    return SAGECAL_OK;
}

int enqueue_mstep(int N, bool scalar, const CompressWorkspace& w, const double* Scc_k, sagecal_c128* J0,
                  sagecal_c128* Jk, int n_trial, bool init, double tau, double* cost_out, double* trace_out,
                  cudaStream_t st) {
    MstepArgs A;
    A.g = make_mgeom(N, choose_pb(N));
    A.lpb = ilog2(A.g.PB);
    A.Src = w.Src; A.Scc = Scc_k;
    A.Ppart = w.Ppart; A.Qpart = w.Qpart; A.cost_cta = w.cost_cta; A.pred_st = w.pred_st; A.mm_st = w.mm_st; A.Htry = w.Htry;
    A.G = w.G; A.M = w.M; A.J_try = w.J_try; A.J0 = J0; A.Jk = Jk;
    A.ctl = w.ctl; A.bar = w.bar; A.n_trial = n_trial; A.init = init ? 1 : 0; A.tau = tau;
    A.cost_out = cost_out; A.trace_out = trace_out;
    int cap = 0, rc;
    if ((rc = scalar ? max_coresident<true>(&cap) : max_coresident<false>(&cap))) return rc;
    int grid = A.g.ntiles < cap ? A.g.ntiles : cap;
    if (grid > MS_MAX_GRID) grid = MS_MAX_GRID;
    if (grid < 1) grid = 1;
    SGC_CUDA(cudaMemsetAsync(w.bar, 0, 256, st));
    void* args[] = {(void*)&A};
    const size_t smem = scalar ? mstep_smem_bytes<true>() : mstep_smem_bytes<false>();
    LaunchScope ls(KK_MSTEP, st);
    SGC_CUDA(cudaLaunchCooperativeKernel(scalar ? (const void*)mstep_kernel<true> : (const void*)mstep_kernel<false>,
                                         dim3((unsigned)grid), dim3(MS_THREADS), args, smem, st));
    return SAGECAL_OK;
}

}  // namespace sgc

using namespace sgc;

// Host-side replay of the M-step kernel's tiling, lane mapping and record lists (CPU tests, no device needed).
extern "C" int sagecal_debug_mstep_cover(int N, int32_t* cover, int64_t* info) {
    if (N < 2 || !cover || !info) return SAGECAL_EINVAL;
    const MGeom g = make_mgeom(N, choose_pb(N));
    const int PB = g.PB, lpb = ilog2(PB);
    const size_t nP = (size_t)g.nqt * N, nQ = (size_t)g.npb * N;
    // bit 0: written, bit 1: carries a baseline, bit 2: read by the station reduction
    unsigned char* fp = new unsigned char[nP]();
    unsigned char* fq = new unsigned char[nQ]();
    int bad = (1 << lpb) == PB ? 0 : 64;
    int64_t seen = 0;
    for (int tile = 0; tile < g.ntiles; tile++) {
        int qt = 0, pb = tile;
        while (qt < g.nqt) {
            const int nl = (g.qmax(qt) + PB - 1) >> lpb;
            if (pb < nl) break;
            pb -= nl; qt++;
        }
        if (qt >= g.nqt || pb >= g.npb) { bad |= 16; continue; }
        seen++;
        for (int warp = 0; warp < MS_WARPS; warp++) {
            const int sq = warp & 3, rg = warp >> 2;
            for (int step = 0; step < PB / 2; step++) {
                const int r = 2 * step + rg, p = (pb << lpb) + r;
                if (p >= N - 1) continue;
                // the staged range of this row must hold every baseline the lanes touch
                const int q0 = MS_TQ * qt, qlo = q0 > p + 1 ? q0 : p + 1, qhi = q0 + MS_TQ < N ? q0 + MS_TQ : N;
                fp[(size_t)qt * N + p] |= 1;
                for (int qi = 0; qi < 8; qi++) {
                    const int q = q0 + 8 * sq + qi;
                    if (q < N && q > p) {
                        if (q < qlo || q >= qhi) bad |= 128;
                        cover[bl_index(N, p, q)]++;
                        fp[(size_t)qt * N + p] |= 2;
                        fq[(size_t)pb * N + q] |= 2;
                    }
                }
            }
        }
        for (int c = 0; c < MS_TQ; c++)
            if (MS_TQ * qt + c < N) fq[(size_t)pb * N + MS_TQ * qt + c] |= 1;
    }
    for (int s = 0; s < N; s++) {
        if (s <= N - 2)
            for (int qt = (s + 1) / MS_TQ; qt < g.nqt; qt++) fp[(size_t)qt * N + s] |= 4;
        if (s >= 1) {
            const int nl = (g.qmax(s / MS_TQ) + PB - 1) >> lpb;
            for (int pb = 0; pb < nl; pb++) {
                if (pb >= g.npb) { bad |= 32; break; }
                fq[(size_t)pb * N + s] |= 4;
            }
        }
    }
    for (size_t x = 0; x < nP; x++) {
        if ((fp[x] & 4) && !(fp[x] & 1)) bad |= 1;   // read but never written
        if ((fp[x] & 2) && !(fp[x] & 4)) bad |= 2;   // carries a baseline but is not read
    }
    for (size_t x = 0; x < nQ; x++) {
        if ((fq[x] & 4) && !(fq[x] & 1)) bad |= 4;
        if ((fq[x] & 2) && !(fq[x] & 4)) bad |= 8;
    }
    delete[] fp;
    delete[] fq;
    info[0] = g.nqt; info[1] = g.npb; info[2] = seen; info[3] = g.B; info[4] = PB; info[5] = g.ntiles;
    return bad;
}
