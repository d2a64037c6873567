// One chunk of a compressed M-step as ONE cooperative kernel (formulas: compress.cuh): the initial
// evaluation at the centre Jones and n_trial Levenberg-Marquardt trial steps, each = cost / gradient / per-station
// J^H J from the per-baseline statistics (rows 8a-4, 8a-5 of SURVEY.md §8(a) re-associated), with the damping,
// accept/reject and 2x2 solves on the device and grid-wide barriers between the phases:
//
//   A  baselines : one THREAD per baseline.  A warp owns a chunk of m consecutive row stations p of one 32-wide
//                  column segment for the whole launch; lane <-> column station q, whose Jones (trial, centre,
//                  difference, Gram matrix) and whose sums (G_q, M_q) stay in registers over the chunk's rows.
//                  The statistics of a row (32 records) are staged in shared memory with cp.async: once per launch
//                  when the warp's rows fit its slots (every N <= 256, and N <= 512 with scalar coherencies), else
//                  one row ahead of the arithmetic through two slots.  Row-station sums (G_p, M_p): a halving
//                  exchange over the lanes (16 additions per row instead of 60), one record per row.  Column-station
//                  sums: one record per (chunk, column).  Cost: one sum per CTA.
//      -- grid barrier --
//   B  control   : every station-owning warp adds the CTA costs and the CTAs' predicted reductions in the same fixed
//                  order (identical everywhere), takes the accept/reject decision and updates mu, nu.  Warp <->
//                  station: adds the station's records (all loads in flight together, one halving exchange; the
//                  CTA's idle warps help as a team when a station has many column records), commits or discards the
//                  trial, solves dJ_p = G_p (M_p + mu I)^-1, writes the next trial Jones; the predicted reduction
//                  is summed per CTA.
//      -- grid barrier --
//
// No atomics in the sums, fixed summation order: bit-reproducible for a given grid.  mstep_kernel: cooperative launch,
// all CTAs co-resident, the grid barrier is an arrive counter in device memory (one red.release per CTA, relaxed
// polling, one acquire fence: 1.25 us at 148 CTAs, measured against cooperative_groups' grid.sync() at 1.2 us, which
// however makes every warp invalidate its L1, and against one-flag-per-CTA schemes at 2.5 us); everything that crosses
// CTAs is read with ld.cg (L2).  mstep_cluster_kernel (N <= 64): one thread-block cluster, the same two phases with
// every exchange in distributed shared memory and the hardware cluster barrier.
#include <math.h>
#include <mutex>
#include <cooperative_groups.h>
#include "compress.cuh"

namespace sgc {

struct MstepArgs {
    MGeom g;
    int slots;                 // shared-memory slots per warp: >= g.m (statistics resident) or 2 (streamed)
    const double *Src, *Scc;
    double *Ppart, *Qpart, *cost_cta, *pred_cta, *mm_cta;
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
__device__ __forceinline__ cplx cadd(cplx a, cplx b) { return mk(a.re + b.re, a.im + b.im); }
__device__ __forceinline__ cplx csub(cplx a, cplx b) { return mk(a.re - b.re, a.im - b.im); }
__device__ __forceinline__ cplx lds_c(const double* p) {
    const double2 v = *reinterpret_cast<const double2*>(p);
    return mk(v.x, v.y);
}

// every lane of every warp gets the same sum / maximum of n <= MS_MAX_GRID values other CTAs wrote; the loads are a
// separate step so that several sums' loads can be in flight together
struct Strided { double t[MS_MAX_GRID / 32]; };
__device__ __forceinline__ Strided strided_load(const double* p, int n, int lane) {
    Strided r;
#pragma unroll
    for (int u = 0; u < MS_MAX_GRID / 32; u++) {
        const int i = 32 * u + lane;
        r.t[u] = i < n ? __ldcg(p + i) : 0.0;
    }
    return r;
}
__device__ __forceinline__ double strided_partial(const Strided& r) {     // this lane's share, fixed order
    double v = 0.0;
#pragma unroll
    for (int u = 0; u < MS_MAX_GRID / 32; u++) v += r.t[u];
    return v;
}
__device__ __forceinline__ double strided_max(const Strided& r) {
    double v = 0.0;
#pragma unroll
    for (int u = 0; u < MS_MAX_GRID / 32; u++) v = fmax(v, r.t[u]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

// ---- grid barrier: an arrive counter, generation gen = 1, 2, ... (the counter is zeroed before every launch) -------
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

// One slot = the statistics of one unit: 32 Src records (lane l's at l * SRC_B: a quarter-warp's 16-byte reads fall
// into 8 different bank groups for both record sizes, 272 = 2*128 + 16 and 80), then 32 Scc records.  The 128-byte Scc
// record of the 2x2 form would put all lanes on one bank group: its eight 16-byte parts are stored rotated by the
// lane index instead.
template <bool SCALAR> struct Slot {
    static constexpr int SRC_B = (SCALAR ? NSRC_SCALAR : NSRC_FULL) * 8;          // 80 / 272
    static constexpr int SCC_B = (SCALAR ? NSCC_SCALAR : NSCC_FULL) * 8;          // 8 / 128
    static constexpr int SCC_OFF = 32 * SRC_B;
    static constexpr int BYTES = 32 * (SRC_B + SCC_B);                            // 2816 / 12800
};
constexpr int MS_CLUSTER_CTAS = 16;   // the largest thread-block cluster (non-portable size)
constexpr int PJ_DOUBLES = 24;    // per warp: J_try (8), J0 (8), D = J_try - J0 (8) of the row station

template <bool SCALAR>
__host__ __device__ constexpr size_t mstep_smem_bytes(int slots) {
    return (size_t)MS_WARPS * slots * Slot<SCALAR>::BYTES + sizeof(double) * (MS_WARPS * PJ_DOUBLES + 3 * MS_WARPS);
}
template <bool SCALAR>
constexpr int max_slots() {   // of the 227 KB a CTA can have
    return (int)((227 * 1024 - sizeof(double) * (MS_WARPS * PJ_DOUBLES + 3 * MS_WARPS)) / ((size_t)MS_WARPS * Slot<SCALAR>::BYTES));
}

// cp.async the statistics of unit (qt, p) into `slot`; the lanes of the warp share the 16-byte chunks
template <bool SCALAR>
__device__ __forceinline__ void issue_unit(const MstepArgs& A, unsigned char* slot, int qt, int p, int lane) {
    using S = Slot<SCALAR>;
    const int N = A.g.N;
    const int q0 = MS_TQ * qt;
    const int qlo = max(q0, p + 1), qhi = min(q0 + MS_TQ, N), cnt = qhi - qlo, l0 = qlo - q0;
    if (cnt <= 0) return;
    const int64_t b0 = bl_index(N, p, qlo);
    const unsigned char* gs = reinterpret_cast<const unsigned char*>(A.Src) + (size_t)b0 * S::SRC_B;
    const unsigned char* gc = reinterpret_cast<const unsigned char*>(A.Scc) + (size_t)b0 * S::SCC_B;
    unsigned char* dc = slot + S::SCC_OFF;
    if (cnt == MS_TQ) {
        // a full row (every unit above the diagonal block): fixed trip counts, offsets are immediates
        constexpr int NCH = MS_TQ * S::SRC_B / 16;                  // 16-byte chunks of the 32 Src records
#pragma unroll
        for (int k = 0; k < NCH / 32; k++) cp_async16(slot + 16 * lane + 512 * k, gs + 16 * lane + 512 * k);
        if (NCH % 32 && lane < NCH % 32) cp_async16(slot + 16 * lane + 512 * (NCH / 32), gs + 16 * lane + 512 * (NCH / 32));
        if (SCALAR) {
            cp_async8(dc + 8 * lane, gc + 8 * lane);
        } else {
            // chunk c = lane + 32 k: record (lane >> 3) + 4 k, part lane & 7, rotated by the record index
            const int rec = lane >> 3, rot0 = ((lane & 7) + rec) & 7;
            unsigned char* d0 = dc + rec * 128 + rot0 * 16;
            unsigned char* d1 = dc + rec * 128 + ((rot0 + 4) & 7) * 16;
#pragma unroll
            for (int k = 0; k < 8; k++) cp_async16(((k & 1) ? d1 : d0) + 512 * k, gc + 16 * lane + 512 * k);
        }
        return;
    }
    {
        unsigned char* d = slot + l0 * S::SRC_B;
        const int nchunk = cnt * (S::SRC_B / 16);
        for (int c = lane; c < nchunk; c += 32) cp_async16(d + 16 * c, gs + 16 * c);
    }
    if (SCALAR) {
        if (lane < cnt) cp_async8(dc + 8 * (l0 + lane), gc + 8 * lane);
    } else {
        for (int c = lane; c < cnt * 8; c += 32) {
            const int l = l0 + (c >> 3);
            cp_async16(dc + l * 128 + (((c & 7) + l) & 7) * 16, gc + 16 * c);
        }
    }
}

// ---- one baseline -------------------------------------------------------------------------------------------------
// The lane's column station q, constant over the rows of its chunk.
struct QSide {
    cplx j[4], d[4];            // J_q (trial), D_q = J_q - J0_q
    double h00, h11; cplx h01;  // J_q^H J_q
};
__device__ __forceinline__ void gram22(const cplx* j, double& h00, double& h11, cplx& h01) {
    h00 = cabs2(j[2], cabs2(j[0], 0.0));
    h11 = cabs2(j[3], cabs2(j[1], 0.0));
    h01 = cfmaca(j[2], j[3], cfmaca(j[0], j[1], mk(0.0, 0.0)));
}

// src / scc: this baseline's staged statistics; pj: the row station's J_try (8 doubles), J0 (8), D (8), warp-uniform
// shared memory.  v[0..7] = this baseline's part of G_p, v[8..11] of M_p (M00, M11, Re M01, Im M01); gq / mq += the
// column station's; cost += the baseline's cost.
template <bool SCALAR>
__device__ __forceinline__ void baseline_task(const double* src, const unsigned char* scc, int lane, const double* pj,
                                              const QSide& Q, double* v, cplx* gq, double* mq, double& cost) {
    double hp00, hp11; cplx hp01;
    {
        const cplx jp[4] = {lds_c(pj), lds_c(pj + 2), lds_c(pj + 4), lds_c(pj + 6)};
        gram22(jp, hp00, hp11, hp01);
    }
    cplx gp[4] = {mk(0.0, 0.0), mk(0.0, 0.0), mk(0.0, 0.0), mk(0.0, 0.0)};
    double acc = 0.0;
    if (SCALAR) {
        const double s2 = *reinterpret_cast<const double*>(scc);
#pragma unroll
        for (int a = 0; a < 4; a++) {
            const int i = a >> 1, j = a & 1;
            const cplx jp[2] = {lds_c(pj + 4 * i), lds_c(pj + 4 * i + 2)};
            const cplx jp0[2] = {lds_c(pj + 8 + 4 * i), lds_c(pj + 8 + 4 * i + 2)};
            const cplx dp[2] = {lds_c(pj + 16 + 4 * i), lds_c(pj + 16 + 4 * i + 2)};
            const cplx sr = lds_c(src + 2 * a);
            // dP[(i,j)] = sum_k D_p[i,k] conj(J_q[j,k]) + J0_p[i,k] conj(D_q[j,k])   (= D_p J0_q^H + J_p D_q^H)
            cplx dP = cmulc(dp[0], Q.j[2 * j]);
            dP = cfmac(dp[1], Q.j[2 * j + 1], dP);
            dP = cfmac(jp0[0], Q.d[2 * j], dP);
            dP = cfmac(jp0[1], Q.d[2 * j + 1], dP);
            const cplx se = mk(fma(-s2, dP.re, sr.re), fma(-s2, dP.im, sr.im));
            acc = fma(dP.re, sr.re + se.re, fma(dP.im, sr.im + se.im, acc));
            gp[2 * i] = cfma(se, Q.j[2 * j], gp[2 * i]);              // G_p[i,k] += Se[(i,j)] J_q[j,k]
            gp[2 * i + 1] = cfma(se, Q.j[2 * j + 1], gp[2 * i + 1]);
            gq[2 * j] = cfmac(jp[0], se, gq[2 * j]);                  // G_q[j,l] += conj(Se[(i,j)]) J_p[i,l]
            gq[2 * j + 1] = cfmac(jp[1], se, gq[2 * j + 1]);
        }
        cost += src[NSRC_SCALAR - 2] - acc;
        v[8] = s2 * Q.h00; v[9] = s2 * Q.h11; v[10] = s2 * Q.h01.re; v[11] = s2 * Q.h01.im;
        mq[0] = fma(s2, hp00, mq[0]); mq[1] = fma(s2, hp11, mq[1]);
        mq[2] = fma(s2, hp01.re, mq[2]); mq[3] = fma(s2, hp01.im, mq[3]);
    } else {
        // Hermitian Scc, packed: (S00, S11) (S22, S33) S01 S02 S03 S12 S13 S23, part t at ((t + lane) & 7) * 16
        cplx S[4][4];
        {
            auto part = [&](int t) { return *reinterpret_cast<const double2*>(scc + (((t + lane) & 7) << 4)); };
            const double2 d0 = part(0), d1 = part(1);
            S[0][0] = mk(d0.x, 0.0); S[1][1] = mk(d0.y, 0.0); S[2][2] = mk(d1.x, 0.0); S[3][3] = mk(d1.y, 0.0);
            const double2 s01 = part(2), s02 = part(3), s03 = part(4), s12 = part(5), s13 = part(6), s23 = part(7);
            S[0][1] = mk(s01.x, s01.y); S[0][2] = mk(s02.x, s02.y); S[0][3] = mk(s03.x, s03.y);
            S[1][2] = mk(s12.x, s12.y); S[1][3] = mk(s13.x, s13.y); S[2][3] = mk(s23.x, s23.y);
        }
#pragma unroll
        for (int x = 0; x < 4; x++) {
#pragma unroll
            for (int y = x + 1; y < 4; y++) S[y][x] = mk(S[x][y].re, -S[x][y].im);
        }
#pragma unroll
        for (int a = 0; a < 4; a++) {
            const int i = a >> 1, j = a & 1;
            const cplx jp[2] = {lds_c(pj + 4 * i), lds_c(pj + 4 * i + 2)};
            // row a of dW: dW[(k,l)] = D_p[i,k] conj(J_q[j,l]) + J0_p[i,k] conj(D_q[j,l])
            // (= D_p (x) conj(J0_q) + J_p (x) conj(D_q), with J0_q = J_q - D_q substituted: no centre Jones per lane)
            cplx dW[4];
            {
                const cplx dp[2] = {lds_c(pj + 16 + 4 * i), lds_c(pj + 16 + 4 * i + 2)};
                const cplx jp0[2] = {lds_c(pj + 8 + 4 * i), lds_c(pj + 8 + 4 * i + 2)};
#pragma unroll
                for (int c = 0; c < 4; c++)
                    dW[c] = cfmac(jp0[c >> 1], Q.d[2 * j + (c & 1)], cmulc(dp[c >> 1], Q.j[2 * j + (c & 1)]));
            }
            // row a of Src (64 B), Sec = Src - dW Scc (the diagonal of Scc is real), cost
            cplx sec[4];
#pragma unroll
            for (int c = 0; c < 4; c++) {
                const cplx sv = lds_c(src + 8 * a + 2 * c);
                cplx t = mk(fma(-dW[c].re, S[c][c].re, sv.re), fma(-dW[c].im, S[c][c].re, sv.im));
#pragma unroll
                for (int d = 0; d < 4; d++)
                    if (d != c) t = cfms(dW[d], S[d][c], t);
                sec[c] = t;
                acc = fma(dW[c].re, sv.re + t.re, fma(dW[c].im, sv.im + t.im, acc));
            }
            // G_p[i,k] += sum_l J_q[j,l] Sec[(i,j),(k,l)];   G_q[j,l] += sum_k J_p[i,k] conj(Sec[(i,j),(k,l)])
            gp[2 * i] = cfma(Q.j[2 * j + 1], sec[1], cfma(Q.j[2 * j], sec[0], gp[2 * i]));
            gp[2 * i + 1] = cfma(Q.j[2 * j + 1], sec[3], cfma(Q.j[2 * j], sec[2], gp[2 * i + 1]));
            gq[2 * j] = cfmac(jp[1], sec[2], cfmac(jp[0], sec[0], gq[2 * j]));
            gq[2 * j + 1] = cfmac(jp[1], sec[3], cfmac(jp[0], sec[1], gq[2 * j + 1]));
        }
        cost += src[NSRC_FULL - 2] - acc;
        // M_p[k,k'] = sum_{l,l'} Hq[l,l'] S[(k,l)][(k',l')]
        v[8] = fma(Q.h00, S[0][0].re, fma(Q.h11, S[1][1].re, 2.0 * fma(Q.h01.re, S[0][1].re, -Q.h01.im * S[0][1].im)));
        v[9] = fma(Q.h00, S[2][2].re, fma(Q.h11, S[3][3].re, 2.0 * fma(Q.h01.re, S[2][3].re, -Q.h01.im * S[2][3].im)));
        {   // M_p[0,1] = Hq00 S[0][2] + Hq01 S[0][3] + conj(Hq01) S[1][2] + Hq11 S[1][3]
            cplx m = mk(Q.h00 * S[0][2].re, Q.h00 * S[0][2].im);
            m = cfma(Q.h01, S[0][3], m);
            m = cfmaca(Q.h01, S[1][2], m);
            v[10] = fma(Q.h11, S[1][3].re, m.re);
            v[11] = fma(Q.h11, S[1][3].im, m.im);
        }
        // M_q[l,l'] = sum_{k,k'} Hp[k,k'] conj(S[(k,l)][(k',l')])
        mq[0] += fma(hp00, S[0][0].re, fma(hp11, S[2][2].re, 2.0 * fma(hp01.re, S[0][2].re, hp01.im * S[0][2].im)));
        mq[1] += fma(hp00, S[1][1].re, fma(hp11, S[3][3].re, 2.0 * fma(hp01.re, S[1][3].re, hp01.im * S[1][3].im)));
        {   // M_q[0,1] = Hp00 conj(S[0][1]) + Hp01 conj(S[0][3]) + conj(Hp01) S[1][2] + Hp11 conj(S[2][3])
            cplx m = mk(hp00 * S[0][1].re, -hp00 * S[0][1].im);
            m = cfmac(hp01, S[0][3], m);
            m = cfmaca(hp01, S[1][2], m);
            mq[2] += fma(hp11, S[2][3].re, m.re);
            mq[3] += fma(-hp11, S[2][3].im, m.im);
        }
    }
#pragma unroll
    for (int x = 0; x < 4; x++) { v[2 * x] = gp[x].re; v[2 * x + 1] = gp[x].im; }
}

// Sum of v[0..15] over the 32 lanes by halving: after step k a lane keeps the half of its values its lane bit selects
// and adds the partner's.  On return v[0] of lane l is the warp total of index 8 b4 + 4 b3 + 2 b2 + b1 (b = bits of
// l; lanes l and l^1 hold the same value).  16 additions per lane, fixed order.
template <int H>
__device__ __forceinline__ void halve_step(double* v, bool up, int mask) {
#pragma unroll
    for (int x = 0; x < H; x++) {
        const double send = up ? v[x] : v[x + H], keep = up ? v[x + H] : v[x];
        v[x] = keep + __shfl_xor_sync(0xffffffffu, send, mask);
    }
}
__device__ __forceinline__ int halve_index(int lane) { return (lane >> 1) & 15; }
__device__ __forceinline__ void halve_sum16(double* v, int lane) {
    halve_step<8>(v, lane & 16, 16);
    halve_step<4>(v, lane & 8, 8);
    halve_step<2>(v, lane & 4, 4);
    halve_step<1>(v, lane & 2, 2);
    v[0] += __shfl_xor_sync(0xffffffffu, v[0], 1);
}

// ---- phase A ------------------------------------------------------------------------------------------------------
struct Smem {
    unsigned char* stage;     // [MS_WARPS][slots][Slot::BYTES]
    double* pj;               // [MS_WARPS][PJ_DOUBLES]
    double* s_red;            // [3][MS_WARPS]: cost, predicted reduction, max diag M per warp
};

struct WarpWork { int chunk, qt, p0, cnt; };     // cnt = 0: this warp has no chunk

// fill the warp's row-station record: lanes 0..3 bring J_try[p], lanes 4..7 J0[p]
__device__ __forceinline__ cplx pj_fetch(const sagecal_c128* jt, const sagecal_c128* j0, int p, int lane) {
    return lane < 8 ? ldcg_c((lane < 4 ? jt : j0) + 4 * p + (lane & 3)) : mk(0.0, 0.0);
}
__device__ __forceinline__ void pj_store(double* pj, cplx mine, int lane) {
    const cplx other = mk(__shfl_down_sync(0xffffffffu, mine.re, 4), __shfl_down_sync(0xffffffffu, mine.im, 4));
    if (lane < 8) { pj[2 * lane] = mine.re; pj[2 * lane + 1] = mine.im; }
    if (lane < 4) { pj[16 + 2 * lane] = mine.re - other.re; pj[16 + 2 * lane + 1] = mine.im - other.im; }
}

// e: evaluation index; at e = 0 the trial point is the centre (Jk, not yet copied to J_try / J0 by everyone).
// seq: running unit counter of the streamed staging (slot = seq & 1), carried over the evaluations.
template <bool SCALAR>
__device__ __forceinline__ void phase_baselines(const MstepArgs& A, const Smem& sm, const WarpWork& ww, int e, bool last,
                                                const cplx* j0q, int& seq) {
    using S = Slot<SCALAR>;
    const MGeom& g = A.g;
    const int N = g.N;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const bool resident = A.slots >= g.m;
    double cost = 0.0;
    if (ww.cnt > 0) {
        const sagecal_c128* jt_src = e == 0 ? A.Jk : A.J_try;
        const sagecal_c128* j0_src = e == 0 ? A.Jk : A.J0;
        const int q = MS_TQ * ww.qt + lane;
        const bool qlive = q < N;
        unsigned char* wstage = sm.stage + (size_t)warp * A.slots * S::BYTES;
        double* pj = sm.pj + warp * PJ_DOUBLES;
        cplx pnext = pj_fetch(jt_src, j0_src, ww.p0, lane);
        QSide Q;
#pragma unroll
        for (int x = 0; x < 4; x++) {
            Q.j[x] = e == 0 ? j0q[x] : (qlive ? ldcg_c(A.J_try + 4 * q + x) : mk(0.0, 0.0));
            Q.d[x] = csub(Q.j[x], j0q[x]);
        }
        gram22(Q.j, Q.h00, Q.h11, Q.h01);
        cplx gq[4] = {mk(0.0, 0.0), mk(0.0, 0.0), mk(0.0, 0.0), mk(0.0, 0.0)};
        double mq[4] = {0.0, 0.0, 0.0, 0.0};
        for (int r = 0; r < ww.cnt; r++) {
            const int p = ww.p0 + r;
            const unsigned char* slot;
            if (resident) {
                slot = wstage + (size_t)r * S::BYTES;
                if (e == 0 && r == 0) { cp_async_wait<0>(); __syncwarp(); }
            } else {
                // the next unit in the running order (the first row of the next evaluation after the last row)
                const bool more = r + 1 < ww.cnt || !last;
                if (more) issue_unit<SCALAR>(A, wstage + (size_t)((seq + 1) & 1) * S::BYTES, ww.qt, r + 1 < ww.cnt ? p + 1 : ww.p0, lane);
                cp_async_commit();
                cp_async_wait<1>();
                __syncwarp();
                slot = wstage + (size_t)(seq & 1) * S::BYTES;
                seq++;
            }
            pj_store(pj, pnext, lane);
            __syncwarp();
            if (r + 1 < ww.cnt) pnext = pj_fetch(jt_src, j0_src, p + 1, lane);
            double v[16];
#pragma unroll
            for (int x = 0; x < 16; x++) v[x] = 0.0;
            if (qlive && q > p)
                baseline_task<SCALAR>(reinterpret_cast<const double*>(slot + lane * S::SRC_B),
                                      slot + S::SCC_OFF + lane * S::SCC_B, lane, pj, Q, v, gq, mq, cost);
            halve_sum16(v, lane);
            const int idx = halve_index(lane);
            if (!(lane & 1) && idx < MS_NV) A.Ppart[(size_t)(g.ubase(ww.qt) + p) * MS_NV + idx] = v[0];
            __syncwarp();                                           // pj and (streamed) the slot are rewritten next
        }
        double2* out = reinterpret_cast<double2*>(A.Qpart + ((size_t)ww.chunk * MS_TQ + lane) * MS_NV);
        out[0] = make_double2(gq[0].re, gq[0].im); out[1] = make_double2(gq[1].re, gq[1].im);
        out[2] = make_double2(gq[2].re, gq[2].im); out[3] = make_double2(gq[3].re, gq[3].im);
        out[4] = make_double2(mq[0], mq[1]); out[5] = make_double2(mq[2], mq[3]);
    }
    cost = wsum(cost);
    if (lane == 0) sm.s_red[warp] = cost;
}

// ---- phase B helpers ----------------------------------------------------------------------------------------------
struct StAcc { cplx g[4]; cplx m[4]; double x0, x1; };

// Where station s finds its records: as row station one record per column segment that holds a q > s, as column
// station the chunks of its segment that hold a row p < s.  Constant over the launch, computed once per warp for its
// first station (the integer divisions behind cbase() would otherwise sit on the critical path of every evaluation).
struct StationPlan { int s, qt0, nrow, nc; const double* colbase; };
__device__ __forceinline__ StationPlan make_station_plan(const MstepArgs& A, int s) {
    const MGeom& g = A.g;
    StationPlan sp;
    sp.s = s;
    sp.qt0 = (s + 1) / MS_TQ;
    sp.nrow = s <= g.N - 2 ? g.nqt - sp.qt0 : 0;
    const int qts = s / MS_TQ, c0 = g.cbase(qts);
    const int nr = min(s, g.nrows(qts));
    sp.nc = (nr + g.m - 1) / g.m;
    sp.colbase = A.Qpart + ((size_t)c0 * MS_TQ + (s - MS_TQ * qts)) * MS_NV;
    return sp;
}

// Adds the station's records, lanes over records (the loads of up to five records per lane are issued before the first
// addition), then ONE halving exchange sums the 12 station values together with two more lane-partial values x0, x1
// (the CTA costs and predicted reductions: the same numbers in the same lanes of every warp, so every warp of the grid
// gets bit-identical totals) and 14 shuffles hand every lane every total.
__device__ __forceinline__ void rec_load(const double* base, bool on, double2* t) {
    const double2* rec = reinterpret_cast<const double2*>(base);
#pragma unroll
    for (int x = 0; x < MS_NV / 2; x++) t[x] = on ? __ldcg(rec + x) : make_double2(0.0, 0.0);
}
// A station with many column records (up to one per chunk of its segment: 128 at N = 512, 255 at N = 256) would keep
// its warp busy long after the others are done, and the grid barrier waits for the slowest: when every warp owns at
// most one station, the otherwise idle warps of the CTA join a TEAM (Team: `size` warps, this warp is `member`, member
// 0 owns the station).  The members take the 32-record batches of the column records in turn, each sums its share by
// the same halving exchange, the helpers hand their 12 partial sums over through shared memory and a named barrier of
// the team, and the owner adds them in member order.  Fixed order: bit-reproducible.
struct Team { int size, member, owner_warp, stride; };   // member j of the team is warp owner_warp + j * stride
__device__ __forceinline__ StAcc station_reduce(const MstepArgs& A, const StationPlan& sp, int lane, double x0, double x1,
                                                const Team& tm, double* s_team) {
    const MGeom& g = A.g;
    double acc[16];
#pragma unroll
    for (int x = 0; x < 16; x++) acc[x] = 0.0;
    // the owner's row records (at most one per column segment) and the member's first four column batches are loaded
    // before the first addition
    double2 tr[MS_NV / 2];
    {
        const int qt = sp.qt0 + lane;
        rec_load(A.Ppart + (size_t)(g.ubase(qt < g.nqt ? qt : 0) + sp.s) * MS_NV, tm.member == 0 && lane < sp.nrow, tr);
    }
    for (int b0 = tm.member; 32 * b0 < sp.nc; b0 += 4 * tm.size) {
        double2 tc[4][MS_NV / 2];
#pragma unroll
        for (int u = 0; u < 4; u++) {
            const int c = 32 * (b0 + u * tm.size) + lane;
            rec_load(sp.colbase + (size_t)(c < sp.nc ? c : 0) * MS_TQ * MS_NV, c < sp.nc, tc[u]);
        }
#pragma unroll
        for (int x = 0; x < MS_NV / 2; x++) {
#pragma unroll
            for (int u = 0; u < 4; u++) { acc[2 * x] += tc[u][x].x; acc[2 * x + 1] += tc[u][x].y; }
        }
    }
#pragma unroll
    for (int x = 0; x < MS_NV / 2; x++) { acc[2 * x] += tr[x].x; acc[2 * x + 1] += tr[x].y; }
    if (tm.member == 0) {
        for (int i = 32; i < sp.nrow; i += 32) {          // more than 32 column segments (N > 1024)
            const int qt = sp.qt0 + i + lane;
            rec_load(A.Ppart + (size_t)(g.ubase(qt < g.nqt ? qt : 0) + sp.s) * MS_NV, i + lane < sp.nrow, tr);
#pragma unroll
            for (int x = 0; x < MS_NV / 2; x++) { acc[2 * x] += tr[x].x; acc[2 * x + 1] += tr[x].y; }
        }
        acc[12] = x0; acc[13] = x1;
    }
    halve_sum16(acc, lane);
    const int idx = halve_index(lane);
    if (tm.size > 1) {
        const int id = 1 + tm.owner_warp, cnt = 32 * tm.size;
        if (tm.member > 0) {
            if (!(lane & 1) && idx < MS_NV) s_team[(tm.owner_warp + tm.member * tm.stride) * MS_NV + idx] = acc[0];
            asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(cnt) : "memory");
            return StAcc();
        }
        asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(cnt) : "memory");
        if (idx < MS_NV)
            for (int j = 1; j < tm.size; j++) acc[0] += s_team[(tm.owner_warp + j * tm.stride) * MS_NV + idx];
    }
    double t[14];
#pragma unroll
    for (int x = 0; x < 14; x++) t[x] = __shfl_sync(0xffffffffu, acc[0], 2 * x);     // lane 2x holds index x
    StAcc r;
#pragma unroll
    for (int x = 0; x < 4; x++) r.g[x] = mk(t[2 * x], t[2 * x + 1]);
    r.m[0] = mk(t[8], 0.0); r.m[1] = mk(t[10], t[11]); r.m[2] = mk(t[10], -t[11]); r.m[3] = mk(t[9], 0.0);
    r.x0 = t[12]; r.x1 = t[13];
    return r;
}

// dJ = G (M + mu I)^-1, J_try = J + dJ; writes the trial Jones; returns this station's predicted reduction
// Re tr(G^H dJ) + mu ||dJ||^2
__device__ __forceinline__ double trial_step(const MstepArgs& A, int s, int lane, const cplx* g, const cplx* m,
                                             const cplx* jj, double mu) {
    const double a = m[0].re + mu, d = m[3].re + mu;
    const cplx b = m[1];
    const double det = a * d - (b.re * b.re + b.im * b.im);
    const double rdet = 1.0 / det;
    const cplx inv[4] = {mk(d * rdet, 0.0), mk(-b.re * rdet, -b.im * rdet), mk(-b.re * rdet, b.im * rdet), mk(a * rdet, 0.0)};
    cplx dj[4];
    dj[0] = cfma(g[1], inv[2], cmul(g[0], inv[0]));
    dj[1] = cfma(g[1], inv[3], cmul(g[0], inv[1]));
    dj[2] = cfma(g[3], inv[2], cmul(g[2], inv[0]));
    dj[3] = cfma(g[3], inv[3], cmul(g[2], inv[1]));
    double pred = 0.0;
#pragma unroll
    for (int x = 0; x < 4; x++) {
        pred += g[x].re * dj[x].re + g[x].im * dj[x].im;
        pred += mu * (dj[x].re * dj[x].re + dj[x].im * dj[x].im);
    }
    if (lane == 0) {
#pragma unroll
        for (int x = 0; x < 4; x++) st_c(A.J_try + 4 * s + x, cadd(jj[x], dj[x]));
    }
    return pred;
}

// thread 0 adds (or takes the maximum of) the warps' values in a fixed order and publishes the CTA's
__device__ __forceinline__ void publish(const double* s_w, double* out, bool is_max) {
    double c = s_w[0];
#pragma unroll
    for (int w = 1; w < MS_WARPS; w++) c = is_max ? fmax(c, s_w[w]) : c + s_w[w];
    out[blockIdx.x] = c;
}

template <bool SCALAR>
__global__ void __launch_bounds__(MS_THREADS, 1)
mstep_kernel(const MstepArgs A) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    using S = Slot<SCALAR>;
    Smem sm;
    sm.stage = smem_raw;
    sm.pj = reinterpret_cast<double*>(smem_raw + (size_t)MS_WARPS * A.slots * S::BYTES);
    sm.s_red = sm.pj + MS_WARPS * PJ_DOUBLES;
    const MGeom& g = A.g;
    const int N = g.N;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    // warps are numbered across the CTAs first, so that a small array spreads over many SMs
    const int gw = warp * gridDim.x + blockIdx.x, nw = gridDim.x * MS_WARPS;
    unsigned gen = 0;

    WarpWork ww;
    ww.chunk = gw; ww.qt = 0; ww.p0 = 0; ww.cnt = 0;
    if (gw < g.nchunks) g.decode(gw, ww.qt, ww.p0, ww.cnt);
    const bool resident = A.slots >= g.m;
    int seq = 0;
    cplx j0q[4] = {mk(0.0, 0.0), mk(0.0, 0.0), mk(0.0, 0.0), mk(0.0, 0.0)};
    if (ww.cnt > 0) {
        // the statistics do not depend on the Jones: start their staging right away
        unsigned char* wstage = sm.stage + (size_t)warp * A.slots * S::BYTES;
        if (resident) {
            for (int r = 0; r < ww.cnt; r++) issue_unit<SCALAR>(A, wstage + (size_t)r * S::BYTES, ww.qt, ww.p0 + r, lane);
        } else {
            issue_unit<SCALAR>(A, wstage, ww.qt, ww.p0, lane);
        }
        cp_async_commit();
        const int q = MS_TQ * ww.qt + lane;
        if (q < N) {
#pragma unroll
            for (int x = 0; x < 4; x++) j0q[x] = ldcg_c(A.Jk + 4 * q + x);
        }
    }

    // this warp's stations: gw, gw + nw, ...; the plan of the first (for almost every shape the only one)
    StationPlan sp0;
    sp0.s = gw; sp0.qt0 = 0; sp0.nrow = 0; sp0.nc = 0; sp0.colbase = A.Qpart;
    if (gw < N) sp0 = make_station_plan(A, gw);
    // teams (station_reduce): with at most one station per warp, stations sit on warps 0 .. ns_w-1 of a CTA and the
    // warps above them help: member j of the team of owner warp o is warp o + j * ns_w
    __shared__ double s_team[MS_WARPS * MS_NV];
    Team tm;
    tm.size = 1; tm.member = 0; tm.owner_warp = warp; tm.stride = 1;
    {
        const int ns_w = (N + (int)gridDim.x - 1) / (int)gridDim.x;
        if (nw >= N && ns_w <= MS_WARPS / 2) {
            tm.size = MS_WARPS / ns_w; tm.stride = ns_w; tm.owner_warp = warp % ns_w; tm.member = warp / ns_w;
            if (tm.member > 0) {
                const int ts = tm.owner_warp * (int)gridDim.x + (int)blockIdx.x;      // the team's station
                sp0.s = N;
                if (tm.member < tm.size && ts < N) sp0 = make_station_plan(A, ts);
            }
        }
    }
    const bool owner = tm.member == 0 && sp0.s < N, helper = tm.member > 0 && sp0.s < N;

    // LM state, identical in every thread that owns a station
    double phi = 0.0, mu = A.init ? 0.0 : A.ctl->mu, nu = A.init ? 2.0 : A.ctl->nu;

    // the centre of this chunk's statistics = the current Jones of the cluster (read by the later write-back)
    for (int s = gw; s < N; s += nw)
        if (lane < 4) st_c(A.J0 + 4 * s + lane, ldcg_c(A.Jk + 4 * s + lane));

    for (int e = 0; e <= A.n_trial; e++) {
        const bool last = e == A.n_trial;
        phase_baselines<SCALAR>(A, sm, ww, e, last, j0q, seq);
        __syncthreads();
        if (threadIdx.x == 0) publish(sm.s_red, A.cost_cta, false);
        grid_barrier(A.bar, ++gen);

        // Warps without a station have nothing to decide; they only keep the barriers company.
        double pred_w = 0.0;
        if (e == 0 && A.init) {
            // (phi, G, M) at the centre are the accepted state; mu = tau * max_p max(M_p00, M_p11)
            double mm = 0.0;
            if (helper) station_reduce(A, sp0, lane, 0.0, 0.0, tm, s_team);
            if (owner) {
                const Strided cost_l = strided_load(A.cost_cta, (int)gridDim.x, lane);
                for (int s = sp0.s; s < N; s += nw) {
                    const StAcc r = station_reduce(A, s == sp0.s ? sp0 : make_station_plan(A, s), lane, strided_partial(cost_l), 0.0, tm, s_team);
                    if (lane == 0) {
#pragma unroll
                        for (int x = 0; x < 4; x++) { st_c(A.G + 4 * s + x, r.g[x]); st_c(A.M + 4 * s + x, r.m[x]); }
                    }
                    mm = fmax(mm, fmax(r.m[0].re, r.m[3].re));
                    phi = r.x0;
                }
            }
            if (lane == 0) sm.s_red[2 * MS_WARPS + warp] = mm;
            __syncthreads();
            if (threadIdx.x == 0) publish(sm.s_red + 2 * MS_WARPS, A.mm_cta, true);
            grid_barrier(A.bar, ++gen);
            if (owner) {
                mu = A.tau * strided_max(strided_load(A.mm_cta, (int)gridDim.x, lane));
                nu = 2.0;
                if (!(mu >= 1e-300)) mu = 1e-300;
                if (mu > 1e300) mu = 1e300;
                if (!last) {
                    for (int s = sp0.s; s < N; s += nw) {
                        cplx g4[4], m4[4], jj[4];
#pragma unroll
                        for (int x = 0; x < 4; x++) { g4[x] = ldcg_c(A.G + 4 * s + x); m4[x] = ldcg_c(A.M + 4 * s + x); jj[x] = ldcg_c(A.Jk + 4 * s + x); }
                        pred_w += trial_step(A, s, lane, g4, m4, jj, mu);
                    }
                }
            }
        } else if (helper) {
            station_reduce(A, sp0, lane, 0.0, 0.0, tm, s_team);
        } else if (owner) {
            // All loads are issued before anything is consumed: the CTA partials, the accepted (G, M, J) and the trial
            // J of the station (16 complex numbers: lane x & 15 holds one), then its records.
            const Strided cost_l = strided_load(A.cost_cta, (int)gridDim.x, lane);
            const Strided pred_l = strided_load(A.pred_cta + (size_t)((e + 1) & 1) * MS_MAX_GRID, e > 0 ? (int)gridDim.x : 0, lane);
            const int which = lane & 15;
            auto old_elem = [&](int s) {
                const sagecal_c128* src = which < 4 ? A.G : which < 8 ? A.M : which < 12 ? A.Jk : A.J_try;
                return ldcg_c(src + 4 * s + (which & 3));
            };
            cplx mine = old_elem(sp0.s);
            StAcc r = station_reduce(A, sp0, lane, strided_partial(cost_l), strided_partial(pred_l), tm, s_team);
            const double fresh = r.x0;
            bool accept = false;
            if (e == 0) {
                phi = fresh;                  // re-centre: fresh (phi, G, M) at the accepted Jones, mu and nu continue
            } else {
                // summed per CTA in the previous evaluation; this evaluation's go to the other half
                const double pred = r.x1;
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
            for (int s = sp0.s; s < N; s += nw) {
                if (s != sp0.s) {
                    mine = old_elem(s);
                    r = station_reduce(A, make_station_plan(A, s), lane, 0.0, 0.0, tm, s_team);
                }
                cplx g4[4], m4[4], jj[4];
#pragma unroll
                for (int x = 0; x < 4; x++) {
                    // at e = 0 the trial array is not written yet: the trial point is the current Jones
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
                if (!last) pred_w += trial_step(A, s, lane, g4, m4, jj, mu);
            }
        }
        if (!last) {
            if (lane == 0) sm.s_red[MS_WARPS + warp] = pred_w;
            __syncthreads();
            if (threadIdx.x == 0) publish(sm.s_red + MS_WARPS, A.pred_cta + (size_t)(e & 1) * MS_MAX_GRID, false);
            grid_barrier(A.bar, ++gen);
        }
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        A.ctl->phi = phi; A.ctl->mu = mu; A.ctl->nu = nu;
        if (A.cost_out) *A.cost_out = phi;
        if (A.trace_out) *A.trace_out = phi;
    }
}

// ---- the smallest arrays: ONE thread-block cluster, exchanges through distributed shared memory ---------------------
// N <= 64 (two column segments, at most 94 units): every unit has its own warp in a cluster of up to 16 CTAs and every
// station its own warp, so nothing of an evaluation has to travel through global memory: a warp stores its row record
// and its 32 column records straight into the shared memory of the CTA whose warp owns that station
// (st.shared::cluster through map_shared_rank), the owner sums them from its own shared memory, keeps the accepted
// (G, M, J) of its station in registers for the whole launch and stores the next trial Jones into EVERY CTA's copy of
// the Jones table; cost and predicted reduction go to every CTA as one value per CTA.  Two hardware cluster barriers
// (release / acquire) per evaluation, no L2 round trip on the critical path.  Same sums in the same order as the grid
// form: fixed, bit-reproducible.
constexpr int CL_MAXN = 64, CL_MAXROWS = 63, CL_NQT = 2;
template <bool SCALAR>
__host__ __device__ constexpr size_t mstep_cluster_smem_bytes() {
    return (size_t)MS_WARPS * Slot<SCALAR>::BYTES +
           sizeof(double) * (MS_WARPS * PJ_DOUBLES + 3 * MS_WARPS + 2 * CL_MAXN * 8 + MS_WARPS * CL_NQT * MS_NV +
                             MS_WARPS * CL_MAXROWS * MS_NV + 4 * MS_CLUSTER_CTAS);
}
__device__ __forceinline__ cplx sel4(const cplx* a, int i) { return i == 0 ? a[0] : i == 1 ? a[1] : i == 2 ? a[2] : a[3]; }

template <bool SCALAR>
__global__ void __launch_bounds__(MS_THREADS, 1)
mstep_cluster_kernel(const MstepArgs A) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    using S = Slot<SCALAR>;
    namespace cg = cooperative_groups;
    cg::cluster_group cluster = cg::this_cluster();
    const MGeom& g = A.g;
    const int N = g.N, G = (int)gridDim.x, rank = (int)blockIdx.x;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int gw = warp * G + rank;                      // this warp's unit (m = 1) and its station
    unsigned char* stage = smem_raw + (size_t)warp * S::BYTES;
    double* pj = reinterpret_cast<double*>(smem_raw + (size_t)MS_WARPS * S::BYTES) + warp * PJ_DOUBLES;
    double* s_red = reinterpret_cast<double*>(smem_raw + (size_t)MS_WARPS * S::BYTES) + MS_WARPS * PJ_DOUBLES;
    double* cl_j = s_red + 3 * MS_WARPS;                 // [CL_MAXN][8]  trial Jones, this CTA's copy
    double* cl_j0 = cl_j + CL_MAXN * 8;                  // [CL_MAXN][8]  centre Jones
    double* cl_prow = cl_j0 + CL_MAXN * 8;               // [MS_WARPS][CL_NQT][12]      row records of this CTA's stations
    double* cl_pcol = cl_prow + MS_WARPS * CL_NQT * MS_NV;         // [MS_WARPS][CL_MAXROWS][12] column records
    double* cl_part = cl_pcol + MS_WARPS * CL_MAXROWS * MS_NV;     // [4][MS_CLUSTER_CTAS]: cost, pred (2 halves), max diag M

    int qt = 0, p = 0, cnt = 0;
    if (gw < g.nchunks) g.decode(gw, qt, p, cnt);
    const int q = MS_TQ * qt + lane;
    const bool qlive = q < N, has_unit = cnt > 0, has_station = gw < N;
    if (has_unit) issue_unit<SCALAR>(A, stage, qt, p, lane);
    cp_async_commit();
    // every CTA reads the cluster's current Jones itself: centre and first trial point
    for (int i = threadIdx.x; i < 4 * N; i += MS_THREADS) {
        const cplx z = ldcg_c(A.Jk + i);
        cl_j[2 * i] = z.re; cl_j[2 * i + 1] = z.im;
        cl_j0[2 * i] = z.re; cl_j0[2 * i + 1] = z.im;
        if (rank == 0) st_c(A.J0 + i, z);                // the centre of this chunk's statistics, for the write-back
    }
    // this warp's station: accepted G, M, J and the trial J, one complex number per lane (lane & 15)
    const int which = lane & 15;
    cplx mine = mk(0.0, 0.0);
    if (has_station && which >= 8) mine = ldcg_c(A.Jk + 4 * gw + (which & 3));
    const int nrow = has_station && gw <= N - 2 ? g.nqt - (gw + 1) / MS_TQ : 0;      // its row records: segments qt0 ..
    const int qt0 = (gw + 1) / MS_TQ, qts = gw / MS_TQ;
    const int ncol = has_station ? min(gw, g.nrows(qts)) : 0;                        // its column records: rows p < s
    cp_async_wait<0>();
    __syncthreads();
    cluster.sync();                                      // every CTA is running before anyone stores into it

    cplx j0q[4], jq[4];
#pragma unroll
    for (int x = 0; x < 4; x++) j0q[x] = qlive && has_unit ? lds_c(cl_j0 + 8 * q + 2 * x) : mk(0.0, 0.0);
    double phi = 0.0, mu = A.init ? 0.0 : A.ctl->mu, nu = A.init ? 2.0 : A.ctl->nu;

    for (int e = 0; e <= A.n_trial; e++) {
        const bool last = e == A.n_trial;
        // ---- phase A: this warp's unit ----
        double cost = 0.0;
        if (has_unit) {
            QSide Q;
#pragma unroll
            for (int x = 0; x < 4; x++) {
                jq[x] = qlive ? lds_c(cl_j + 8 * q + 2 * x) : mk(0.0, 0.0);
                Q.j[x] = jq[x];
                Q.d[x] = csub(jq[x], j0q[x]);
            }
            gram22(Q.j, Q.h00, Q.h11, Q.h01);
            if (lane < 8) {                              // the row station's J_try (lanes 0..3), J0 (4..7), D
                const cplx a = lds_c((lane < 4 ? cl_j : cl_j0) + 8 * p + 2 * (lane & 3));
                pj[2 * lane] = a.re; pj[2 * lane + 1] = a.im;
                if (lane < 4) { const cplx b = lds_c(cl_j0 + 8 * p + 2 * lane); pj[16 + 2 * lane] = a.re - b.re; pj[17 + 2 * lane] = a.im - b.im; }
            }
            __syncwarp();
            cplx gq[4] = {mk(0.0, 0.0), mk(0.0, 0.0), mk(0.0, 0.0), mk(0.0, 0.0)};
            double mq[4] = {0.0, 0.0, 0.0, 0.0};
            double v[16];
#pragma unroll
            for (int x = 0; x < 16; x++) v[x] = 0.0;
            if (qlive && q > p)
                baseline_task<SCALAR>(reinterpret_cast<const double*>(stage + lane * S::SRC_B),
                                      stage + S::SCC_OFF + lane * S::SCC_B, lane, pj, Q, v, gq, mq, cost);
            halve_sum16(v, lane);
            const int idx = halve_index(lane);
            if (!(lane & 1) && idx < MS_NV) {            // row record -> the CTA of the warp that owns station p
                double* dst = cluster.map_shared_rank(cl_prow, p % G) + ((p / G) * CL_NQT + qt) * MS_NV;
                dst[idx] = v[0];
            }
            if (qlive) {                                 // column record of row p -> the owner of station q
                double2* dst = reinterpret_cast<double2*>(cluster.map_shared_rank(cl_pcol, q % G) + ((q / G) * CL_MAXROWS + p) * MS_NV);
                dst[0] = make_double2(gq[0].re, gq[0].im); dst[1] = make_double2(gq[1].re, gq[1].im);
                dst[2] = make_double2(gq[2].re, gq[2].im); dst[3] = make_double2(gq[3].re, gq[3].im);
                dst[4] = make_double2(mq[0], mq[1]); dst[5] = make_double2(mq[2], mq[3]);
            }
        }
        cost = wsum(cost);
        if (lane == 0) s_red[warp] = cost;
        __syncthreads();
        if (warp == 0 && lane < G) {                     // the CTA's cost, to every CTA of the cluster
            double c = s_red[0];
#pragma unroll
            for (int w = 1; w < MS_WARPS; w++) c += s_red[w];
            cluster.map_shared_rank(cl_part, lane)[rank] = c;
        }
        cluster.sync();

        // ---- phase B: this warp's station ----
        double pred_w = 0.0, mm = 0.0;
        StAcc r;
        if (has_station) {
            double acc[16];
#pragma unroll
            for (int x = 0; x < 16; x++) acc[x] = 0.0;
            if (lane < nrow) {
                const double* rec = cl_prow + (warp * CL_NQT + qt0 + lane) * MS_NV;
#pragma unroll
                for (int x = 0; x < MS_NV; x++) acc[x] += rec[x];
            }
            for (int c = lane; c < ncol; c += 32) {
                const double* rec = cl_pcol + (warp * CL_MAXROWS + c) * MS_NV;
#pragma unroll
                for (int x = 0; x < MS_NV; x++) acc[x] += rec[x];
            }
            acc[12] = lane < G ? cl_part[lane] : 0.0;
            acc[13] = (e > 0 && lane < G) ? cl_part[(1 + ((e + 1) & 1)) * MS_CLUSTER_CTAS + lane] : 0.0;
            halve_sum16(acc, lane);
            double t[14];
#pragma unroll
            for (int x = 0; x < 14; x++) t[x] = __shfl_sync(0xffffffffu, acc[0], 2 * x);
#pragma unroll
            for (int x = 0; x < 4; x++) r.g[x] = mk(t[2 * x], t[2 * x + 1]);
            r.m[0] = mk(t[8], 0.0); r.m[1] = mk(t[10], t[11]); r.m[2] = mk(t[10], -t[11]); r.m[3] = mk(t[9], 0.0);
            r.x0 = t[12]; r.x1 = t[13];
        }
        bool accept = false, take = false, step = false;
        if (e == 0 && A.init) {
            if (has_station) { phi = r.x0; mm = fmax(r.m[0].re, r.m[3].re); }
            if (lane == 0) s_red[2 * MS_WARPS + warp] = mm;
            __syncthreads();
            if (warp == 0 && lane < G) {
                double c = s_red[2 * MS_WARPS];
#pragma unroll
                for (int w = 1; w < MS_WARPS; w++) c = fmax(c, s_red[2 * MS_WARPS + w]);
                cluster.map_shared_rank(cl_part, lane)[3 * MS_CLUSTER_CTAS + rank] = c;
            }
            cluster.sync();
            double m = lane < G ? cl_part[3 * MS_CLUSTER_CTAS + lane] : 0.0;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
            mu = A.tau * m;
            nu = 2.0;
            take = true; step = !last;
        } else if (has_station) {
            const double fresh = r.x0;
            if (e == 0) {
                phi = fresh;
            } else {
                const double pred = r.x1;
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
            take = accept || e == 0; step = !last;
        }
        if (!(mu >= 1e-300)) mu = 1e-300;
        if (mu > 1e300) mu = 1e300;
        if (nu > 0x1p60) nu = 0x1p60;
        if (has_station) {
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
            // the accepted state stays in registers
            if (which < 4) mine = sel4(g4, which);
            else if (which < 8) mine = sel4(m4, which & 3);
            else if (which < 12) mine = sel4(jj, which & 3);
            if (step) {
                // dJ = G (M + mu I)^-1, J_try = J + dJ
                const double a = m4[0].re + mu, d = m4[3].re + mu;
                const cplx b = m4[1];
                const double rdet = 1.0 / (a * d - (b.re * b.re + b.im * b.im));
                const cplx inv[4] = {mk(d * rdet, 0.0), mk(-b.re * rdet, -b.im * rdet), mk(-b.re * rdet, b.im * rdet), mk(a * rdet, 0.0)};
                cplx dj[4], jt[4];
                dj[0] = cfma(g4[1], inv[2], cmul(g4[0], inv[0]));
                dj[1] = cfma(g4[1], inv[3], cmul(g4[0], inv[1]));
                dj[2] = cfma(g4[3], inv[2], cmul(g4[2], inv[0]));
                dj[3] = cfma(g4[3], inv[3], cmul(g4[2], inv[1]));
#pragma unroll
                for (int x = 0; x < 4; x++) {
                    jt[x] = cadd(jj[x], dj[x]);
                    pred_w += g4[x].re * dj[x].re + g4[x].im * dj[x].im;
                    pred_w += mu * (dj[x].re * dj[x].re + dj[x].im * dj[x].im);
                }
                if (which >= 12) mine = sel4(jt, which & 3);
                // the trial Jones of this station, into every CTA's table: lane -> (CTA lane % G, entries lane / G, ...)
                for (int o = lane; o < 4 * G; o += 32) {
                    const int dst_rank = o % G, x = o / G;
                    const cplx z = sel4(jt, x);
                    double2* dst = reinterpret_cast<double2*>(cluster.map_shared_rank(cl_j, dst_rank) + 8 * gw + 2 * x);
                    *dst = make_double2(z.re, z.im);
                }
            }
        }
        if (!last) {
            if (lane == 0) s_red[MS_WARPS + warp] = pred_w;
            __syncthreads();
            if (warp == 0 && lane < G) {
                double c = s_red[MS_WARPS];
#pragma unroll
                for (int w = 1; w < MS_WARPS; w++) c += s_red[MS_WARPS + w];
                cluster.map_shared_rank(cl_part, lane)[(1 + (e & 1)) * MS_CLUSTER_CTAS + rank] = c;
            }
            cluster.sync();
        }
    }
    if (has_station && lane >= 8 && lane < 12) st_c(A.Jk + 4 * gw + (lane & 3), mine);
    if (rank == 0 && threadIdx.x == 0) {
        A.ctl->phi = phi; A.ctl->mu = mu; A.ctl->nu = nu;
        if (A.cost_out) *A.cost_out = phi;
        if (A.trace_out) *A.trace_out = phi;
    }
    cluster.sync();                                      // nobody leaves while others may still store into it
}

// ---- host side ----------------------------------------------------------------------------------------------------
size_t compress_workspace_bytes(int N, int K, bool scalar) {
    const MGeom g = make_mgeom(N, MS_MAX_WARPS);
    size_t n = 0;
    n += round_up(sizeof(double) * (size_t)(K > 0 ? K : 1) * nscc(scalar) * g.B, 256);
    n += round_up(sizeof(double) * (size_t)nsrc(scalar) * g.B, 256);
    n += round_up(sizeof(double) * (size_t)g.U * MS_NV, 256);
    n += round_up(sizeof(double) * (size_t)MS_MAX_WARPS * MS_TQ * MS_NV, 256);
    n += 4 * round_up(sizeof(double) * MS_MAX_GRID, 256);
    n += 3 * round_up((size_t)N * 64, 256);
    n += 256 + 256;
    n += round_up((size_t)2 * N * 64, 256);
    n += round_up(sizeof(double) * (size_t)GRP * nsrc(scalar) * g.B, 256);
    n += round_up(sizeof(double) * (size_t)ngroups(K > 0 ? K : 1) * GRP_PAIRS * nxg(scalar) * g.B, 256);
    n += round_up((size_t)2 * GRP * N * 64, 256);
    return n;
}

CompressWorkspace carve_compress(int N, int K, bool scalar, void* ws) {
    const MGeom g = make_mgeom(N, MS_MAX_WARPS);
    CompressWorkspace w;
    char* p = (char*)ws;
    auto take = [&](size_t n) { char* o = p; p += round_up(n, 256); return o; };
    w.Scc = (double*)take(sizeof(double) * (size_t)(K > 0 ? K : 1) * nscc(scalar) * g.B);
    w.Src = (double*)take(sizeof(double) * (size_t)nsrc(scalar) * g.B);
    w.Ppart = (double*)take(sizeof(double) * (size_t)g.U * MS_NV);
    w.Qpart = (double*)take(sizeof(double) * (size_t)MS_MAX_WARPS * MS_TQ * MS_NV);
    w.cost_cta = (double*)take(sizeof(double) * MS_MAX_GRID);
    w.pred_cta = (double*)take(sizeof(double) * 2 * MS_MAX_GRID);
    w.mm_cta = (double*)take(sizeof(double) * MS_MAX_GRID);
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

// Launch plan of the M-step kernel for N stations on a device with `sms` SMs (one CTA per SM): work decomposition,
// slots per warp, grid.  Device independent but for `sms` and `cluster_cap` (the largest thread-block cluster the
// device schedules, 0 = none), so that the host replay below sees what the kernel does.

struct MstepPlan { MGeom g; int slots, grid; bool cluster; };
static MstepPlan make_plan(int N, bool scalar, int sms, int cluster_cap) {
    MstepPlan pl;
    int cap = sms < MS_MAX_GRID ? sms : MS_MAX_GRID;
    if (cap < 1) cap = 1;
    while (cap * MS_WARPS < (N + MS_TQ - 1) / MS_TQ) cap++;            // one warp per column segment at the very least
    pl.g = make_mgeom(N, cap * MS_WARPS);
    const int smax = scalar ? max_slots<true>() : max_slots<false>();
    pl.slots = pl.g.m <= smax ? pl.g.m : 2;
    // a small array spreads over many SMs with few warps each (4 busy warps per CTA until every SM has a CTA)
    const int want = (pl.g.nchunks + 3) / 4;
    pl.grid = want < cap ? want : cap;
    if (pl.grid * MS_WARPS < pl.g.nchunks) pl.grid = (pl.g.nchunks + MS_WARPS - 1) / MS_WARPS;
    if (pl.grid < 1) pl.grid = 1;
    // the smallest arrays run as ONE thread-block cluster (mstep_cluster_kernel): a warp per unit, a warp per station
    pl.cluster = N <= CL_MAXN && pl.g.m == 1 && pl.g.nchunks <= cluster_cap * MS_WARPS;
    if (pl.cluster) {
        if (pl.grid > cluster_cap) pl.grid = cluster_cap;
        if (pl.grid * MS_WARPS < pl.g.nchunks) pl.grid = (pl.g.nchunks + MS_WARPS - 1) / MS_WARPS;
    }
    return pl;
}

struct MstepDevice { bool ready; int sms, cluster_cap; };
template <bool SCALAR>
static int mstep_prepare(MstepDevice* out) {
    // per device: the opt-in to large dynamic shared memory is a per-device function attribute
    static MstepDevice devs[64] = {};
    static std::mutex mu;                              // two host threads may meet here on their first call
    std::lock_guard<std::mutex> lk(mu);
    int dev = 0;
    SGC_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return SAGECAL_EUNSUPPORTED;
    MstepDevice& d = devs[dev];
    if (!d.ready) {
        const int smem = (int)mstep_smem_bytes<SCALAR>(max_slots<SCALAR>());
        SGC_CUDA(cudaFuncSetAttribute(mstep_kernel<SCALAR>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        SGC_CUDA(cudaFuncSetAttribute(mstep_cluster_kernel<SCALAR>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                      (int)mstep_cluster_smem_bytes<SCALAR>()));
        SGC_CUDA(cudaDeviceGetAttribute(&d.sms, cudaDevAttrMultiProcessorCount, dev));
        // the largest cluster (16 needs the non-portable opt-in, 8 is portable) that can be resident with the
        // shared memory of a small array (its rows are resident: one slot per warp)
        d.cluster_cap = 0;
        const bool np = cudaFuncSetAttribute(mstep_cluster_kernel<SCALAR>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) == cudaSuccess;
        for (int csz = np ? MS_CLUSTER_CTAS : 8; csz >= 2 && !d.cluster_cap; csz >>= 1) {
            cudaLaunchConfig_t cfg = {};
            cfg.gridDim = dim3((unsigned)csz); cfg.blockDim = dim3(MS_THREADS);
            cfg.dynamicSmemBytes = mstep_cluster_smem_bytes<SCALAR>();
            cudaLaunchAttribute at;
            at.id = cudaLaunchAttributeClusterDimension;
            at.val.clusterDim.x = (unsigned)csz; at.val.clusterDim.y = 1; at.val.clusterDim.z = 1;
            cfg.attrs = &at; cfg.numAttrs = 1;
            int ncl = 0;
            if (cudaOccupancyMaxActiveClusters(&ncl, mstep_cluster_kernel<SCALAR>, &cfg) == cudaSuccess && ncl >= 1) d.cluster_cap = csz;
        }
        (void)cudaGetLastError();
        d.ready = true;
    }
    *out = d;
    return SAGECAL_OK;
}

int enqueue_mstep(int N, bool scalar, const CompressWorkspace& w, const double* Scc_k, sagecal_c128* J0,
                  sagecal_c128* Jk, int n_trial, bool init, double tau, double* cost_out, double* trace_out,
                  cudaStream_t st) {
    MstepDevice dv;
    int rc;
    if ((rc = scalar ? mstep_prepare<true>(&dv) : mstep_prepare<false>(&dv))) return rc;
    const MstepPlan pl = make_plan(N, scalar, dv.sms, dv.cluster_cap);
    if (pl.grid > dv.sms || pl.grid > MS_MAX_GRID) return SAGECAL_EUNSUPPORTED;     // more column segments than warps
    MstepArgs A;
    A.g = pl.g;
    A.slots = pl.slots;
    A.Src = w.Src; A.Scc = Scc_k;
    A.Ppart = w.Ppart; A.Qpart = w.Qpart; A.cost_cta = w.cost_cta; A.pred_cta = w.pred_cta; A.mm_cta = w.mm_cta;
    A.G = w.G; A.M = w.M; A.J_try = w.J_try; A.J0 = J0; A.Jk = Jk;
    A.ctl = w.ctl; A.bar = w.bar; A.n_trial = n_trial; A.init = init ? 1 : 0; A.tau = tau;
    A.cost_out = cost_out; A.trace_out = trace_out;
    const size_t smem = scalar ? mstep_smem_bytes<true>(pl.slots) : mstep_smem_bytes<false>(pl.slots);
    if (pl.cluster) {
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)pl.grid); cfg.blockDim = dim3(MS_THREADS);
        cfg.dynamicSmemBytes = scalar ? mstep_cluster_smem_bytes<true>() : mstep_cluster_smem_bytes<false>();
        cfg.stream = st;
        cudaLaunchAttribute at;
        at.id = cudaLaunchAttributeClusterDimension;
        at.val.clusterDim.x = (unsigned)pl.grid; at.val.clusterDim.y = 1; at.val.clusterDim.z = 1;
        cfg.attrs = &at; cfg.numAttrs = 1;
        LaunchScope ls(KK_MSTEP, st);
        if (scalar) SGC_CUDA(cudaLaunchKernelEx(&cfg, mstep_cluster_kernel<true>, A));
        else SGC_CUDA(cudaLaunchKernelEx(&cfg, mstep_cluster_kernel<false>, A));
        return SAGECAL_OK;
    }
    SGC_CUDA(cudaMemsetAsync(w.bar, 0, 256, st));
    void* args[] = {(void*)&A};
    LaunchScope ls(KK_MSTEP, st);
    SGC_CUDA(cudaLaunchCooperativeKernel(scalar ? (const void*)mstep_kernel<true> : (const void*)mstep_kernel<false>,
                                         dim3((unsigned)pl.grid), dim3(MS_THREADS), args, smem, st));
    return SAGECAL_OK;
}

}  // namespace sgc

using namespace sgc;

// Host-side replay of the M-step kernel's work decomposition and record lists (CPU tests, no device needed): the same
// MGeom / make_plan the launch uses, for a device with `sms` SMs.
extern "C" int sagecal_debug_mstep_cover(int N, int sms, int32_t* cover, int64_t* info) {
    if (N < 2 || sms < 1 || !cover || !info) return SAGECAL_EINVAL;
    const MstepPlan pl = make_plan(N, false, sms, sms >= MS_CLUSTER_CTAS ? MS_CLUSTER_CTAS : 0);
    const MGeom& g = pl.g;
    const size_t nP = (size_t)g.U, nQ = (size_t)g.nchunks * MS_TQ;
    // bit 0: written, bit 1: carries a baseline, bit 2: read by the station reduction
    unsigned char* fp = new unsigned char[nP]();
    unsigned char* fq = new unsigned char[nQ]();
    int bad = 0;
    if (g.nchunks > pl.grid * MS_WARPS) bad |= 16;
    int64_t units = 0;
    for (int gw = 0; gw < pl.grid * MS_WARPS; gw++) {
        if (gw >= g.nchunks) continue;
        int qt, p0, cnt;
        g.decode(gw, qt, p0, cnt);
        if (cnt < 1 || cnt > g.m || qt >= g.nqt || p0 + cnt > g.nrows(qt)) { bad |= 16; continue; }
        if (gw != g.cbase(qt) + p0 / g.m) bad |= 32;
        for (int r = 0; r < cnt; r++) {
            const int p = p0 + r;
            const size_t u = (size_t)g.ubase(qt) + p;
            if (u >= nP) { bad |= 32; continue; }
            if (fp[u] & 1) bad |= 64;                   // a unit visited twice
            fp[u] |= 1;
            units++;
            for (int lane = 0; lane < 32; lane++) {
                const int q = MS_TQ * qt + lane;
                if (q < N && q > p) {
                    cover[bl_index(N, p, q)]++;
                    fp[u] |= 2;
                    fq[(size_t)gw * MS_TQ + lane] |= 2;
                }
            }
        }
        for (int lane = 0; lane < 32; lane++) fq[(size_t)gw * MS_TQ + lane] |= 1;
    }
    for (int s = 0; s < N; s++) {
        if (s <= N - 2)
            for (int qt = (s + 1) / MS_TQ; qt < g.nqt; qt++) fp[(size_t)g.ubase(qt) + s] |= 4;
        if (s >= 1) {
            const int qt = s / MS_TQ, c0 = g.cbase(qt);
            const int nr = s < g.nrows(qt) ? s : g.nrows(qt), nc = (nr + g.m - 1) / g.m;
            for (int c = 0; c < nc; c++) fq[(size_t)(c0 + c) * MS_TQ + (s - MS_TQ * qt)] |= 4;
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
    info[0] = g.nqt; info[1] = g.m; info[2] = g.nchunks; info[3] = g.B; info[4] = g.U; info[5] = units;
    info[6] = pl.grid; info[7] = pl.slots;
    return bad;
}
