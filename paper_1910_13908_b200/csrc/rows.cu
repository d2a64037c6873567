// Measurement-set rows <-> the canonical interval layout, and flags (second part:
// "per-row station index arrays (non-canonical order, flags)").
//
// The hot kernels address a sample by arithmetic on (t, p, q, channel) and carry no per-sample mask: that is what
// lets the LM pass keep a station's sums in registers and the compressed M-step walk a baseline's time slots.  A
// general row list is therefore brought INTO that layout once per interval (one gather, HBM-bound: 64 B read + 64 B
// written per sample) instead of teaching every kernel indirection:
//   * row (ant1, ant2, tslot) goes to slot t*B + b(min, max); a row given as (q, p) is the Hermitian transpose of
//     the (p, q) measurement (V_qp = V_pq^H, uvw_qp = -uvw_pq), so it is conjugate-transposed on the way;
//   * a slot no row maps to is flagged; flagged samples are ZERO in the visibilities and (sagecal_apply_flags) in
//     every cluster's coherencies, so E = 0 - J*0*J^H = 0 there: they add nothing to the cost, the gradient, J^H J or
//     the compressed statistics, at no cost to the hot loops;
//   * sagecal_canonical_to_rows hands results (the residual) back in the caller's row order and orientation.
// Index work only; the winner among duplicate rows is fixed (highest row index) so results are run-to-run identical.
#include "common.cuh"

namespace sgc {

constexpr int ROW_THREADS = 256;

__global__ void __launch_bounds__(ROW_THREADS)
rows_slot_kernel(int N, int T, int64_t B, int64_t n, const int32_t* __restrict__ ant1,
                 const int32_t* __restrict__ ant2, const int32_t* __restrict__ tslot, long long* owner,
                 int64_t* __restrict__ row_map, int32_t* status) {
    const int64_t r = (int64_t)blockIdx.x * ROW_THREADS + threadIdx.x;
    if (r >= n) return;
    const int a = ant1[r], b = ant2[r], t = tslot[r];
    int64_t m = -1;
    if (a < 0 || a >= N || b < 0 || b >= N || t < 0 || t >= T) atomicAdd(status + 1, 1);
    else if (a == b) atomicAdd(status + 0, 1);
    else {
        const int p = min(a, b), q = max(a, b);
        const int64_t slot = (int64_t)t * B + bl_index(N, p, q);
        m = 2 * slot + (a > b ? 1 : 0);
        atomicMax(owner + slot, (long long)r);
    }
    row_map[r] = m;
}

// rows that lost their slot to a later duplicate
__global__ void __launch_bounds__(ROW_THREADS)
rows_resolve_kernel(int64_t n, const long long* __restrict__ owner, int64_t* row_map, int32_t* status) {
    const int64_t r = (int64_t)blockIdx.x * ROW_THREADS + threadIdx.x;
    if (r >= n) return;
    const int64_t m = row_map[r];
    if (m >= 0 && owner[m >> 1] != r) {
        row_map[r] = -1;
        atomicAdd(status + 2, 1);
    }
}

// [XX, XY, YX, YY] -> its Hermitian transpose
__device__ __forceinline__ void herm(m22& v) {
    const cplx xy = v.a[1];
    v.a[0].im = -v.a[0].im;
    v.a[1] = mk(v.a[2].re, -v.a[2].im);
    v.a[2] = mk(xy.re, -xy.im);
    v.a[3].im = -v.a[3].im;
}

__global__ void __launch_bounds__(ROW_THREADS)
rows_gather_kernel(int F, int64_t samples, const long long* __restrict__ owner, const int32_t* __restrict__ ant1,
                   const int32_t* __restrict__ ant2, const double* __restrict__ uvw_in,
                   const sagecal_c128* __restrict__ vis_in, const uint8_t* __restrict__ flag_in,
                   double* __restrict__ uvw, sagecal_c128* __restrict__ vis, uint8_t* __restrict__ flags,
                   int32_t* status) {
    const int64_t i = (int64_t)blockIdx.x * ROW_THREADS + threadIdx.x;
    if (i >= samples) return;
    const int64_t slot = i / F;
    const int c = (int)(i - slot * F);
    const long long src = owner[slot];
    m22 v;
    v.a[0] = v.a[1] = v.a[2] = v.a[3] = mk(0.0, 0.0);
    uint8_t fl = 1;
    double u0 = 0.0, u1 = 0.0, u2 = 0.0;
    if (src >= 0) {
        const bool sw = ant1[src] > ant2[src];
        fl = flag_in ? (flag_in[(size_t)src * F + c] != 0) : 0;
        if (!fl) {
            load_m22_stream(vis_in + ((size_t)src * F + c) * 4, v);
            if (sw) herm(v);
        }
        if (c == 0) {
            const double s = sw ? -1.0 : 1.0;
            u0 = s * uvw_in[3 * src]; u1 = s * uvw_in[3 * src + 1]; u2 = s * uvw_in[3 * src + 2];
        }
    } else if (c == 0) {
        atomicAdd(status + 3, 1);
    }
    store_m22(vis + 4 * i, v);
    flags[i] = fl;
    if (c == 0) { uvw[3 * slot] = u0; uvw[3 * slot + 1] = u1; uvw[3 * slot + 2] = u2; }
}

__global__ void __launch_bounds__(ROW_THREADS)
rows_scatter_kernel(int F, int64_t n_samples, const int64_t* __restrict__ row_map,
                    const sagecal_c128* __restrict__ vis_c, sagecal_c128* __restrict__ vis_out) {
    const int64_t i = (int64_t)blockIdx.x * ROW_THREADS + threadIdx.x;
    if (i >= n_samples) return;
    const int64_t r = i / F;
    const int c = (int)(i - r * F);
    const int64_t m = row_map[r];
    if (m < 0) return;
    m22 v;
    load_m22_stream(vis_c + ((size_t)(m >> 1) * F + c) * 4, v);
    if (m & 1) herm(v);
    store_m22(vis_out + 4 * i, v);
}

template <bool SCALAR>
__global__ void __launch_bounds__(ROW_THREADS)
apply_flags_kernel(int64_t samples, int K, const uint8_t* __restrict__ flags, sagecal_c128* __restrict__ coh,
                   sagecal_c128* __restrict__ vis) {
    const int64_t i = (int64_t)blockIdx.x * ROW_THREADS + threadIdx.x;
    if (i >= samples || !flags[i]) return;
    if (vis) { stg256(vis + 4 * i, 0.0, 0.0, 0.0, 0.0); stg256(vis + 4 * i + 2, 0.0, 0.0, 0.0, 0.0); }
    for (int k = 0; k < K; k++) {
        if (SCALAR) {
            coh[(size_t)k * samples + i].re = 0.0;
            coh[(size_t)k * samples + i].im = 0.0;
        } else {
            sagecal_c128* p = coh + ((size_t)k * samples + i) * 4;
            stg256(p, 0.0, 0.0, 0.0, 0.0);
            stg256(p + 2, 0.0, 0.0, 0.0, 0.0);
        }
    }
}

static inline unsigned blocks_for(int64_t n) { return (unsigned)((n + ROW_THREADS - 1) / ROW_THREADS); }

}  // namespace sgc

using namespace sgc;

extern "C" size_t sagecal_rows_workspace_bytes(int N, int T) {
    if (N < 2 || T < 1) return 0;
    return round_up(sizeof(long long) * (size_t)T * ((size_t)N * (N - 1) / 2), 256);
}

extern "C" int sagecal_rows_to_canonical(int N, int T, int F, int64_t nrows_in, const int32_t* ant1,
                                         const int32_t* ant2, const int32_t* tslot, const double* uvw_in,
                                         const sagecal_c128* vis_in, const uint8_t* flag_in, double* uvw,
                                         sagecal_c128* vis, uint8_t* flags, int64_t* row_map, int32_t* status,
                                         void* workspace, size_t workspace_bytes, void* stream) {
    if (N < 2 || T < 1 || F < 1 || nrows_in < 0) return SAGECAL_EINVAL;
    if (!uvw || !vis || !flags || !status || !aligned(vis, 32)) return SAGECAL_EINVAL;
    if (nrows_in > 0 && (!ant1 || !ant2 || !tslot || !uvw_in || !vis_in || !row_map || !aligned(vis_in, 32)))
        return SAGECAL_EINVAL;
    if (!workspace || !aligned(workspace, 256) || workspace_bytes < sagecal_rows_workspace_bytes(N, T))
        return SAGECAL_EWORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    const int64_t B = (int64_t)N * (N - 1) / 2, slots = (int64_t)T * B, samples = slots * F;
    long long* owner = (long long*)workspace;
    SGC_CUDA(cudaMemsetAsync(owner, 0xFF, sizeof(long long) * (size_t)slots, st));   // -1
    SGC_CUDA(cudaMemsetAsync(status, 0, 4 * sizeof(int32_t), st));
    if (nrows_in > 0) {
        {
            LaunchScope ls(KK_ROWS, st);
            rows_slot_kernel<<<blocks_for(nrows_in), ROW_THREADS, 0, st>>>(N, T, B, nrows_in, ant1, ant2, tslot, owner, row_map, status);
            SGC_LAUNCH_CHECK();
        }
        {
            LaunchScope ls(KK_ROWS, st);
            rows_resolve_kernel<<<blocks_for(nrows_in), ROW_THREADS, 0, st>>>(nrows_in, owner, row_map, status);
            SGC_LAUNCH_CHECK();
        }
    }
    LaunchScope ls(KK_ROWS, st);
    rows_gather_kernel<<<blocks_for(samples), ROW_THREADS, 0, st>>>(F, samples, owner, ant1, ant2, uvw_in, vis_in, flag_in, uvw, vis, flags, status);
    SGC_LAUNCH_CHECK();
    return SAGECAL_OK;
}

extern "C" int sagecal_canonical_to_rows(int N, int T, int F, int64_t nrows_in, const int64_t* row_map,
                                         const sagecal_c128* vis_canonical, sagecal_c128* vis_out, void* stream) {
    if (N < 2 || T < 1 || F < 1 || nrows_in < 0) return SAGECAL_EINVAL;
    if (nrows_in == 0) return SAGECAL_OK;
    if (!row_map || !vis_canonical || !vis_out || vis_canonical == vis_out || !aligned(vis_canonical, 32) || !aligned(vis_out, 32))
        return SAGECAL_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    LaunchScope ls(KK_ROWS, st);
    rows_scatter_kernel<<<blocks_for(nrows_in * F), ROW_THREADS, 0, st>>>(F, nrows_in * F, row_map, vis_canonical, vis_out);
    SGC_LAUNCH_CHECK();
    return SAGECAL_OK;
}

extern "C" int sagecal_apply_flags(int N, int T, int F, int K, const uint8_t* flags, int coh_format,
                                   sagecal_c128* coh, sagecal_c128* vis, void* stream) {
    if (N < 2 || T < 1 || F < 1 || K < 0 || !flags) return SAGECAL_EINVAL;
    if (coh_format != SAGECAL_COH_FULL && coh_format != SAGECAL_COH_SCALAR) return SAGECAL_EINVAL;
    if (K > 0 && (!coh || !aligned(coh, coh_format == SAGECAL_COH_SCALAR ? 16 : 32))) return SAGECAL_EINVAL;
    if (vis && !aligned(vis, 32)) return SAGECAL_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const int64_t samples = (int64_t)T * ((int64_t)N * (N - 1) / 2) * F;
    LaunchScope ls(KK_ROWS, st);
    if (coh_format == SAGECAL_COH_SCALAR) apply_flags_kernel<true><<<blocks_for(samples), ROW_THREADS, 0, st>>>(samples, K, flags, coh, vis);
    else apply_flags_kernel<false><<<blocks_for(samples), ROW_THREADS, 0, st>>>(samples, K, flags, coh, vis);
    SGC_LAUNCH_CHECK();
    return SAGECAL_OK;
}
