// transform.cu — AO->MO two-step half transform (DESIGN.md steps A1, A2):
//   A1  H^P_{i nu} = sum_mu C_{mu i} (P|mu nu)        (P|mu nu) streamed from packed mu>=nu storage
//   A2  B^P_{ia}   = sum_nu H^P_{i nu} C_{nu a}       written as B[a][i][P], aux index contiguous
// DF form of the cluster integral projection, PAPER.md Eq. S49 (L526).
//
// Kernels: unpack (packed triangle -> square, HBM-bound), transpose (tiny), and one persistent
// TMA + mbarrier + DMMA GEMM  C = A * B^T  over K-major operands (see mma_pipeline.cuh), used for both
// half transforms with an output-column remap that lands B directly in its final [a][i][P] layout.
#include "mma_pipeline.cuh"
#include "sie_internal.h"
#include "../../include/sie_dfmp2.h"

namespace sie {

// ------------------------------------------------------------------------------------------------
__global__ void transpose_kernel(const double* __restrict__ in, int rows, int cols, double* __restrict__ out, int ld_out) {
    __shared__ double tile[32][33];
    const int r0 = blockIdx.y * 32, c0 = blockIdx.x * 32;
    for (int rr = threadIdx.y; rr < 32; rr += 8) {
        const int r = r0 + rr, c = c0 + threadIdx.x;
        tile[rr][threadIdx.x] = (r < rows && c < cols) ? in[(size_t)r * cols + c] : 0.0;
    }
    __syncthreads();
    for (int rr = threadIdx.y; rr < 32; rr += 8) {
        const int c = c0 + rr, r = r0 + threadIdx.x;
        if (c < cols && r < rows) out[(size_t)c * ld_out + r] = tile[threadIdx.x][rr];
    }
}

int launch_transpose(const double* in, int rows, int cols, double* out, int ld_out, cudaStream_t st) {
    dim3 grid((cols + 31) / 32, (rows + 31) / 32), block(32, 8);
    transpose_kernel<<<grid, block, 0, st>>>(in, rows, cols, out, ld_out);
    note_launch();
    cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? SIE_OK : set_cuda_error(e);
}

// ------------------------------------------------------------------------------------------------
// packed (mu >= nu, idx = mu(mu+1)/2 + nu) -> full symmetric matrix; grid (tc, tr, P), only tr >= tc works.
__global__ void unpack_kernel(const double* __restrict__ Lp, int nao, double* __restrict__ Lfull, int ld) {
    const int tc = blockIdx.x, tr = blockIdx.y;
    if (tc > tr) return;
    __shared__ double tile[32][33];
    const size_t npair = (size_t)nao * (nao + 1) / 2;
    const double* src = Lp + (size_t)blockIdx.z * npair;
    double* dst = Lfull + (size_t)blockIdx.z * nao * ld;
    for (int rr = threadIdx.y; rr < 32; rr += 8) {
        const int mu = tr * 32 + rr, nu = tc * 32 + threadIdx.x;
        double x = 0.0;
        if (mu < nao && nu <= mu) {
            x = __ldg(src + (size_t)mu * (mu + 1) / 2 + nu);
            dst[(size_t)mu * ld + nu] = x;
        }
        tile[rr][threadIdx.x] = x;
    }
    __syncthreads();
    for (int rr = threadIdx.y; rr < 32; rr += 8) {
        const int nu = tc * 32 + rr, mu = tr * 32 + threadIdx.x;  // element (mu,nu) of the tile, written at [nu][mu]
        if (mu < nao && nu < mu) dst[(size_t)nu * ld + mu] = tile[threadIdx.x][rr];
    }
}

int launch_unpack(const double* Lp, int np, int nao, double* Lfull, int ld, cudaStream_t st) {
    const int nt = (nao + 31) / 32;
    for (int z0 = 0; z0 < np; z0 += 65535) {
        const int nz = (np - z0 < 65535) ? np - z0 : 65535;
        dim3 grid(nt, nt, nz), block(32, 8);
        unpack_kernel<<<grid, block, 0, st>>>(Lp + (size_t)z0 * ((size_t)nao * (nao + 1) / 2), nao,
                                              Lfull + (size_t)z0 * nao * ld, ld);
        note_launch();
    }
    cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? SIE_OK : set_cuda_error(e);
}

// ------------------------------------------------------------------------------------------------
template <class Cfg>
__global__ void __launch_bounds__(Cfg::NTHREADS, 1)
gemm_tn_kernel(const __grid_constant__ CUtensorMap mapA, const __grid_constant__ CUtensorMap mapB, int m_tiles, int n_tiles,
               int nb_inner, long long inner_pad, int kblocks, GemmOut out) {
    extern __shared__ unsigned char smem_dyn[];
    unsigned char* smem = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(smem_dyn) + 127) & ~uintptr_t(127));
    double* stages = reinterpret_cast<double*>(smem);
    uint64_t* full = reinterpret_cast<uint64_t*>(smem + Cfg::STAGES * Cfg::STAGE_BYTES);
    uint64_t* empty = full + Cfg::STAGES;

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    pipeline_init<Cfg>(full, empty, tid);
    __syncthreads();

    const int ntiles = m_tiles * n_tiles;
    PipeState ps;
    if (warp == Cfg::NCONS) {
        if (lane == 0) {
            tma_prefetch_desc(&mapA);
            tma_prefetch_desc(&mapB);
            for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
                const int mb = tile % m_tiles, nb = tile / m_tiles;
                produce_tile<Cfg>(stages, full, empty, kblocks, ps, &mapA, mb * Cfg::TM, 0, &mapB, (nb % nb_inner) * Cfg::TN,
                                  nb / nb_inner, (uint32_t)Cfg::STAGE_BYTES);
            }
        }
        return;
    }
    const int wm = warp % Cfg::NWM, wn = warp / Cfg::NWM;
    const int g = lane >> 2, t = lane & 3;
    double acc[Cfg::MT][Cfg::NT][2];
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const int mb = tile % m_tiles, nb = tile / m_tiles;
        consume_tile<Cfg>(acc, stages, full, empty, kblocks, ps, wm, wn, lane);
        const long long n_base = (long long)(nb / nb_inner) * inner_pad + (long long)(nb % nb_inner) * Cfg::TN;
#pragma unroll
        for (int j = 0; j < Cfg::NT; ++j) {
            const long long n0 = n_base + wn * Cfg::WN + 8 * j + 2 * t;
            const long long n1 = n0 + 1;
            const long long q0 = n0 / out.inner, r0 = n0 % out.inner;
            const long long q1 = n1 / out.inner, r1 = n1 % out.inner;
            const bool ok0 = n0 < out.n_lin_total && r0 < out.valid_inner;
            const bool ok1 = n1 < out.n_lin_total && r1 < out.valid_inner;
            const long long off0 = q0 * out.stride_outer + r0;
            const long long off1 = q1 * out.stride_outer + r1;
#pragma unroll
            for (int i = 0; i < Cfg::MT; ++i) {
                const int m = mb * Cfg::TM + wm * Cfg::WM + 8 * i + g;
                if (m >= out.M) continue;
                double* p = out.base + (long long)m * out.ld_m;
                if (ok0 && ok1 && off1 == off0 + 1 && ((reinterpret_cast<uintptr_t>(p + off0) & 15) == 0)) {
                    *reinterpret_cast<double2*>(p + off0) = make_double2(acc[i][j][0], acc[i][j][1]);
                } else {
                    if (ok0) p[off0] = acc[i][j][0];
                    if (ok1) p[off1] = acc[i][j][1];
                }
            }
        }
    }
}

template <class Cfg>
static int launch_gemm_cfg(const CUtensorMap& mapA, const CUtensorMap& mapB, int m_tiles, int n_tiles, int nb_inner,
                           long long inner_pad, int kblocks, const GemmOut& out, int num_sms, cudaStream_t st) {
    const size_t smem = (size_t)Cfg::STAGES * Cfg::STAGE_BYTES + 2 * Cfg::STAGES * sizeof(uint64_t) + 128;
    auto kern = gemm_tn_kernel<Cfg>;
    static SmemAttrOnce once;  // per instantiation, per device inside
    const int rc = ensure_smem_attr(reinterpret_cast<const void*>(kern), (int)smem, once);
    if (rc != SIE_OK) return rc;
    const long long ntiles = (long long)m_tiles * n_tiles;
    if (ntiles <= 0) return SIE_OK;
    const int grid = (int)(ntiles < num_sms ? ntiles : num_sms);
    kern<<<grid, Cfg::NTHREADS, smem, st>>>(mapA, mapB, m_tiles, n_tiles, nb_inner, inner_pad, kblocks, out);
    note_launch();
    cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? SIE_OK : set_cuda_error(e);
}

int gemm_tm_for(int m) { return m <= 16 ? 16 : m <= 32 ? 32 : m <= 64 ? 64 : 128; }

int launch_gemm_tn(int tm_sel, const CUtensorMap& mapA, const CUtensorMap& mapB, int m_tiles, int n_tiles, int nb_inner,
                   long long inner_pad, int kblocks, const GemmOut& out, int num_sms, cudaStream_t st) {
    switch (tm_sel) {
        case 16:
            return launch_gemm_cfg<TileCfg<16, 16, 1, 8, 8>>(mapA, mapB, m_tiles, n_tiles, nb_inner, inner_pad, kblocks, out, num_sms, st);
        case 32:
            return launch_gemm_cfg<TileCfg<32, 16, 1, 8, 8>>(mapA, mapB, m_tiles, n_tiles, nb_inner, inner_pad, kblocks, out, num_sms, st);
        case 64:
            return launch_gemm_cfg<TileCfg<32, 32, 2, 4, 8>>(mapA, mapB, m_tiles, n_tiles, nb_inner, inner_pad, kblocks, out, num_sms, st);
        default:
            return launch_gemm_cfg<TileCfg<64, 32, 2, 4, 8>>(mapA, mapB, m_tiles, n_tiles, nb_inner, inner_pad, kblocks, out, num_sms, st);
    }
}

}  // namespace sie
