// Geometry and partial-sum layout of the fused LM evaluation pass (lm_pass.cu), shared with the calibration
// driver (calibrate.cu).  DESIGN.md §5.3.
#pragma once
#include "common.cuh"

namespace sgc {

constexpr int PASS_THREADS = 128;            // one thread per sample slot of a tile segment
constexpr int PASS_WARPS = PASS_THREADS / 32;
constexpr int PASS_NV = 12;                  // doubles per station side: G (4 complex) + M (M00, M11, Re M01, Im M01)
constexpr int PASS_BREC = 26;                // tensor-core form: doubles per baseline record: G_p (8), G_q (8), M_p (4), M_q (4), cost, pad

// The upper triangle of the N x N station grid is cut into column tiles of TQ stations (q) and single rows (p).
// A "unit" is (column c, row p, time chunk tc): TQ*F samples per time slot, contiguous in memory at fixed t.
// Units are enumerated column-major, (p, tc) inside a column, and split evenly over the CTAs ("slots").
struct PassGeom {
    int N, T, F;
    int TQ;      // stations per column tile: max(1, 128/F)
    int nchunk;  // 128-sample chunks per segment: ceil(TQ*F/128) (1 unless F > 128)
    int ncols;   // ceil(N/TQ)
    int TC;      // time chunks per row
    int tlen;    // time slots per chunk
    int nslots;  // CTAs
    int64_t R;   // total (column,row) pairs
    int64_t U;   // total units = R*TC
    int64_t B;   // baselines

    // rows p of column c: 0 <= p < qhi(c)-1
    __host__ __device__ int qhi(int c) const { int h = TQ * (c + 1); return h < N ? h : N; }
    // number of (column,row) pairs in columns < c  (valid for 0 <= c <= ncols-1; all those columns are full)
    __host__ __device__ int64_t cum(int c) const { return (int64_t)TQ * c * (c + 1) / 2 - c; }
    __host__ __device__ int64_t slot_begin(int i) const { return U * (int64_t)i / nslots; }
    // slot that owns unit u
    __host__ __device__ int slot_of(int64_t u) const {
        int i = (int)(((u + 1) * (int64_t)nslots - 1) / U);   // smallest i with slot_begin(i+1) > u  (then fix up)
        if (i < 0) i = 0;
        if (i > nslots - 1) i = nslots - 1;
        while (i > 0 && slot_begin(i) > u) i--;
        while (i < nslots - 1 && slot_begin(i + 1) <= u) i++;
        return i;
    }
    // column of the (column,row) pair index ru
    __host__ __device__ int col_of(int64_t ru) const {
        // largest c in [0, ncols-1] with cum(c) <= ru
        double a = 0.5 * TQ, bq = 0.5 * TQ - 1.0;  // cum(c) = a c^2 + bq c
        int c = (int)((-bq + sqrt(bq * bq + 4.0 * a * (double)ru)) / (2.0 * a));
        if (c < 0) c = 0;
        if (c > ncols - 1) c = ncols - 1;
        while (c > 0 && cum(c) > ru) c--;
        while (c < ncols - 1 && cum(c + 1) <= ru) c++;
        return c;
    }
};

// Workspace layout of one pass (all doubles):
//   Ppart [U][PASS_WARPS][12]   per-unit, per-warp p-side sums (row station p)
//   Pcost [U][PASS_WARPS]       per-unit, per-warp cost
//   Qpart [nslots+ncols][TQ][12] per-(slot,column) q-side sums; record index = slot + column
//   Brec  [B][PASS_BREC]        tensor-core form (2x2 coherencies, lm_pass_mma.cu): one record per baseline
struct PassWorkspace {
    double* Ppart;
    double* Pcost;
    double* Qpart;
    double* Brec;
    double* cost_st;    // [N] tensor-core form: cost of each station's row-role records
    unsigned* counter;  // ticket counter of the reduction's last-block step
};

PassGeom make_pass_geom(int N, int T, int F);
size_t pass_workspace_bytes(const PassGeom& g);
PassWorkspace carve_pass_workspace(const PassGeom& g, void* ws);

// enqueue: partial sums of (cost, G, M) for one cluster at `jones`, then the fixed-order station reduction.
int enqueue_pass(const PassGeom& g, const PassWorkspace& w, const sagecal_c128* x, int coh_format,
                 const sagecal_c128* coh_k, const sagecal_c128* jones, double* cost, sagecal_c128* grad,
                 sagecal_c128* jtj, cudaStream_t st);

// 2x2 coherencies: the same sums on the FP64 tensor cores, one warp per baseline (lm_pass_mma.cu)
int enqueue_pass_mma(const PassGeom& g, const PassWorkspace& w, const sagecal_c128* x, const sagecal_c128* coh_k,
                     const sagecal_c128* jones, double* cost, sagecal_c128* grad, sagecal_c128* jtj, cudaStream_t st);

}  // namespace sgc
