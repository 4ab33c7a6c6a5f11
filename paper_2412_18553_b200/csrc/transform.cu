// transform.cu — AO->MO two-step half transform (DESIGN.md steps A1, A2):
//   A1  H^P_{i nu} = sum_mu C_{mu i} (P|mu nu)        (P|mu nu) streamed from packed mu>=nu storage
//   A2  B^P_{ia}   = sum_nu H^P_{i nu} C_{nu a}       written as B[a][i][P], aux index contiguous
// DF form of the cluster integral projection, PAPER.md Eq. S49 (L526).
//
// Kernels: transposes of the coefficient matrices (tiny) and ONE grouped persistent mbarrier-pipelined DMMA GEMM
// C = A * Bop^T over K-major operands, used for both half transforms of every cluster of a call in one launch per
// stage: A1 gathers its Bop operand straight from the packed triangle (no unpacked square in HBM), A2 lands B directly
// in its final [a][i][P] layout through an output-column remap.
#include <algorithm>
#include <cstring>

#include "mma_pipeline.cuh"
#include "sie_internal.h"
#include "../../include/sie_dfmp2.h"

namespace sie {

// ------------------------------------------------------------------------------------------------
// Grouped persistent GEMM of the transform stages:  C[m][n] = sum_k A[m][k] * Bop[n][k]  for a LIST of jobs in one launch.
//
//   A1 (PACKED = true):  H[i][(P,nu)] = sum_mu CoT[i][mu] * Lsym^P[nu][mu]      A = CoT (TMA), Bop = the PACKED triangle
//   A2 (PACKED = false): B[a][(i,P)]  = sum_nu CvT[a][nu] * H[(i,P)][nu]        A = CvT (TMA), Bop = H (TMA)
//
// A CTA tile is (8*m8) x 128 with m8 <= 16 taken EXACTLY from the job (o = 120 -> 15 m-tiles, no padding to 128; a
// v of 136 is cut into two chunks of 72 rows), 8 consumer warps in a 2 x 4 grid: the warp row wm owns ceil/floor(m8/2)
// m-tiles, every warp 4 n-tiles, and the two warps of one SM sub-partition sit on different warp rows, so the
// sub-partitions issue the same DMMA count.  The per-warp m-tile count is a template parameter behind a warp-uniform switch
// (a predicated-off DMMA would still take its pipe slot).
//
// Operand feed, two K-blocks of 8 per stage (one barrier round trip per 16 k values), each as dense [row][8] lines of 64 B (conflict-free LDS.128, see mma_pipeline.cuh):
//   * A and the TMA-mode Bop: cp.async.bulk.tensor boxes {8, rows, 1}, completion by complete_tx on the stage's `full`.
//   * the packed Bop: (P|mu nu) is stored as lower triangles, row mu at offset mu(mu+1)/2 — only 8-byte aligned and not
//     a TMA tensor, so the producer warps gather it with 8-byte cp.async straight from the packed array: element
//     (n = (P,nu), k = mu) comes from Lp[P][max(mu,nu)(max+1)/2 + min(mu,nu)].  Below the diagonal that is 64 contiguous
//     bytes per row, above it 32-byte runs of 4 consecutive nu; the shared-memory side is always 256 contiguous bytes per
//     warp instruction.  Completion by cp.async.mbarrier.arrive.noinc on the same `full` barrier.  The square
//     (P|mu nu) is never materialised: every packed element is read by the two output tiles that need it, close together
//     in time (the tiles of one P are consecutive in the work list), so it comes from HBM once and from L2 once.
constexpr int XG_NCONS = 8;                 // consumer warps (2 x 4)
#ifndef SIE_XG_NPROD
#define SIE_XG_NPROD 4
#endif
constexpr int XG_NPROD = SIE_XG_NPROD;      // producer warps (4: at small M the gather's address arithmetic is issue-bound on 2)
constexpr int XG_RG = XG_NPROD * 4;         // row groups of the packed gather: thread (k, rg) owns column k of rows rg, rg + XG_RG, ...
constexpr int XG_RPT = 128 / XG_RG;         // rows per producer thread and K-block
constexpr int XG_THREADS = (XG_NCONS + XG_NPROD) * 32;
constexpr int XG_TN = 128, XG_KB = 8, XG_TMMAX = 128;
constexpr int XG_NSUB = 2;                  // K-blocks per pipeline stage: one full/empty barrier round trip per 16 k values
constexpr int XG_STAGES = 6;
constexpr int XG_SUB_DOUBLES = (XG_TMMAX + XG_TN) * XG_KB;   // one K-block: A rows [128][8], then Bop rows [128][8]
constexpr int XG_STAGE_DOUBLES = XG_NSUB * XG_SUB_DOUBLES;
constexpr size_t XG_SMEM = (size_t)XG_STAGES * XG_STAGE_DOUBLES * 8 + 2 * XG_STAGES * 8 + 128;

__device__ __forceinline__ void cp_async_8(uint32_t dst, const double* src, bool valid) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(dst), "l"(src), "r"(valid ? 8 : 0) : "memory");
}
__device__ __forceinline__ void cp_async_arrive_noinc(uint64_t* bar) {
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}

template <int MTW>
__device__ __forceinline__ void xg_consume(double (&acc)[8][4][2], const double* __restrict__ stages, uint64_t* full, uint64_t* empty,
                                           int kblocks, PipeState& ps, int row0, int wn, int lane) {
    const int g = lane >> 2, t = lane & 3;
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
    const uint32_t base = smem_u32(stages);
    const uint32_t offA = base + 8u * (uint32_t)((row0 + g) * XG_KB + 2 * t);
    const uint32_t offB = base + 8u * (uint32_t)(XG_TMMAX * XG_KB + (wn * 32 + g) * XG_KB + 2 * t);
    const int ksteps = (kblocks + XG_NSUB - 1) / XG_NSUB;
    for (int ks = 0; ks < ksteps; ++ks) {
        mbar_wait(&full[ps.stage], ps.phase);
        const uint32_t so = (uint32_t)(ps.stage * XG_STAGE_DOUBLES) * 8u;
#pragma unroll
        for (int u = 0; u < XG_NSUB; ++u) {
            double2 a[MTW > 0 ? MTW : 1], b[4];
#pragma unroll
            for (int i = 0; i < MTW; ++i) a[i] = lds128(offA + so + u * (XG_SUB_DOUBLES * 8) + i * (8 * XG_KB * 8));
#pragma unroll
            for (int j = 0; j < 4; ++j) b[j] = lds128(offB + so + u * (XG_SUB_DOUBLES * 8) + j * (8 * XG_KB * 8));
            if (u == XG_NSUB - 1) {
                __syncwarp();
                if (lane == 0) mbar_arrive(&empty[ps.stage]);  // fragments are in registers
                ps.advance<XG_STAGES>();
            }
#pragma unroll
            for (int i = 0; i < MTW; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) dmma884(acc[i][j][0], acc[i][j][1], a[i].x, b[j].x);
#pragma unroll
            for (int i = 0; i < MTW; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) dmma884(acc[i][j][0], acc[i][j][1], a[i].y, b[j].y);
        }
    }
}

template <bool PACKED>
__global__ void __launch_bounds__(XG_THREADS, 1) xform_gemm_kernel(const XJob* __restrict__ jobs, int njobs, int total_tiles) {
    extern __shared__ unsigned char smem_dyn[];
    unsigned char* smem = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(smem_dyn) + 127) & ~uintptr_t(127));
    double* stages = reinterpret_cast<double*>(smem);
    uint64_t* full = reinterpret_cast<uint64_t*>(smem + (size_t)XG_STAGES * XG_STAGE_DOUBLES * 8);
    uint64_t* empty = full + XG_STAGES;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    if (tid == 0) {
        for (int s = 0; s < XG_STAGES; ++s) {
            mbar_init(&full[s], PACKED ? 1 + XG_NPROD * 32 : 1);
            mbar_init(&empty[s], XG_NCONS);
        }
        fence_mbar_init();
    }
    __syncthreads();

    PipeState ps;
    int job = 0;
    if (warp >= XG_NCONS) {
        // ---------------------------------------------------------------- producers
        const int pt = tid - XG_NCONS * 32;  // 0 .. 63
        if (!PACKED && pt != 0) return;
        const int k = pt & 7, rg = pt >> 3;  // packed gather: this thread owns column k of rows rg, rg + 8, ... of a stage
        const CUtensorMap* acquired = nullptr;
        for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x) {
            while (job + 1 < njobs && tile >= jobs[job + 1].tile_begin) ++job;
            const XJob* J = jobs + job;
            const int lt = tile - J->tile_begin;
            const int mb = lt % J->m_tiles, nb = lt / J->m_tiles;
            const int kblocks = J->kblocks, rowsA = 8 * J->m8;
            if (pt == 0 && &J->mapA != acquired) {  // descriptors live in global memory, rewritten by every call
                tma_acquire_desc(&J->mapA);
                if (!PACKED) tma_acquire_desc(&J->mapB);
                acquired = &J->mapA;
            }
            if (PACKED) {
                // the 16 rows (P, nu) of this thread: offset of the packed row of nu, and of the matrix of P
                const int nao = J->nao;
                const long long npair = J->npair;
                long long rowoff[XG_RPT], matoff[XG_RPT];
                int nu[XG_RPT];
#pragma unroll
                for (int j = 0; j < XG_RPT; ++j) {
                    const long long n = (long long)nb * XG_TN + rg + XG_RG * j;
                    const bool ok = n < J->n_total;
                    const unsigned P = ok ? (unsigned)n / (unsigned)nao : 0u;  // the host keeps n_total below 2^31
                    nu[j] = ok ? (int)((unsigned)n - P * (unsigned)nao) : -1;  // -1: row past the end, zero filled
                    matoff[j] = P * npair;
                    rowoff[j] = matoff[j] + (long long)nu[j] * (nu[j] + 1) / 2;
                }
                const double* Lp = J->Lp;
                const int ksteps = (kblocks + XG_NSUB - 1) / XG_NSUB;
                for (int ks = 0; ks < ksteps; ++ks) {
                    mbar_wait(&empty[ps.stage], ps.phase ^ 1u);
                    double* s = stages + ps.stage * XG_STAGE_DOUBLES;
                    if (pt == 0) {
                        mbar_arrive_expect_tx(&full[ps.stage], (uint32_t)(XG_NSUB * rowsA * XG_KB * 8));
#pragma unroll
                        for (int u = 0; u < XG_NSUB; ++u)  // a K-block past the end (odd count) is all zero fill
                            tma_load_3d(s + u * XG_SUB_DOUBLES, &J->mapA, &full[ps.stage], (ks * XG_NSUB + u) * XG_KB, mb * rowsA, 0);
                    }
#pragma unroll
                    for (int u = 0; u < XG_NSUB; ++u) {
                        const int mu = (ks * XG_NSUB + u) * XG_KB + k;
                        const long long trimu = (long long)mu * (mu + 1) / 2;
                        const bool kok = mu < nao;
                        const uint32_t dst = smem_u32(s + u * XG_SUB_DOUBLES + XG_TMMAX * XG_KB) + 8u * (uint32_t)(rg * XG_KB + k);
#pragma unroll
                        for (int j = 0; j < XG_RPT; ++j) {
                            const long long off = mu <= nu[j] ? rowoff[j] + mu : matoff[j] + trimu + nu[j];
                            const bool ok = kok && nu[j] >= 0;
                            cp_async_8(dst + (uint32_t)(XG_RG * j * XG_KB * 8), Lp + (ok ? off : 0), ok);
                        }
                    }
                    cp_async_arrive_noinc(&full[ps.stage]);
                    ps.advance<XG_STAGES>();
                }
            } else {
                const int ksteps = (kblocks + XG_NSUB - 1) / XG_NSUB;
                for (int ks = 0; ks < ksteps; ++ks) {
                    mbar_wait(&empty[ps.stage], ps.phase ^ 1u);
                    double* s = stages + ps.stage * XG_STAGE_DOUBLES;
                    mbar_arrive_expect_tx(&full[ps.stage], (uint32_t)(XG_NSUB * (rowsA + XG_TN) * XG_KB * 8));
#pragma unroll
                    for (int u = 0; u < XG_NSUB; ++u) {
                        const int kk = (J->k0_blocks + ks * XG_NSUB + u) * XG_KB;
                        tma_load_3d(s + u * XG_SUB_DOUBLES, &J->mapA, &full[ps.stage], kk, mb * rowsA, 0);
                        tma_load_3d(s + u * XG_SUB_DOUBLES + XG_TMMAX * XG_KB, &J->mapB, &full[ps.stage], kk, J->b_c1_off + nb * J->b_c1_mul,
                                    nb * J->b_c2_mul);
                    }
                    ps.advance<XG_STAGES>();
                }
            }
        }
        return;
    }
    // -------------------------------------------------------------------- consumers
    // warp = 4 q + s sits on SM sub-partition s; the two warps of a sub-partition take different warp rows
    const int wq = warp >> 2, wsub = warp & 3;
    const int wm = (wq + wsub) & 1, wn = wsub;
    const int g = lane >> 2, t = lane & 3;
    double acc[8][4][2];
    for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x) {
        while (job + 1 < njobs && tile >= jobs[job + 1].tile_begin) ++job;
        const XJob* J = jobs + job;
        const int lt = tile - J->tile_begin;
        const int mb = lt % J->m_tiles, nb = lt / J->m_tiles;
        const int m8 = J->m8, hi = (m8 + 1) >> 1;
        const int mtw = wm == 0 ? hi : m8 - hi;
        const int row0 = wm == 0 ? 0 : 8 * hi;
#define SIE_XG(M) case M: xg_consume<M>(acc, stages, full, empty, J->kblocks, ps, row0, wn, lane); break;
        switch (mtw) {
            SIE_XG(0) SIE_XG(1) SIE_XG(2) SIE_XG(3) SIE_XG(4) SIE_XG(5) SIE_XG(6) SIE_XG(7) SIE_XG(8)
        }
#undef SIE_XG
        const GemmOut out = J->out;
        const long long n_base = (long long)nb * XG_TN + wn * 32;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const long long n0 = n_base + 8 * j + 2 * t, n1 = n0 + 1;
            const long long q0 = n0 / out.inner, r0 = n0 % out.inner;
            const long long q1 = n1 / out.inner, r1 = n1 % out.inner;
            const bool ok0 = n0 < out.n_lin_total && r0 < out.valid_inner;
            const bool ok1 = n1 < out.n_lin_total && r1 < out.valid_inner;
            const long long off0 = q0 * out.stride_outer + r0, off1 = q1 * out.stride_outer + r1;
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                if (i >= mtw) break;
                const int m = mb * 8 * m8 + row0 + 8 * i + g;
                if (m >= out.M) continue;
                double* p = out.base + (long long)m * out.ld_m;
                if (out.accumulate) {
                    if (ok0) p[off0] += acc[i][j][0];
                    if (ok1) p[off1] += acc[i][j][1];
                } else if (ok0 && ok1 && off1 == off0 + 1 && ((reinterpret_cast<uintptr_t>(p + off0) & 15) == 0)) {
                    *reinterpret_cast<double2*>(p + off0) = make_double2(acc[i][j][0], acc[i][j][1]);
                } else {
                    if (ok0) p[off0] = acc[i][j][0];
                    if (ok1) p[off1] = acc[i][j][1];
                }
            }
        }
    }
}

int launch_xform_gemm(bool packed, const XJob* d_jobs, int njobs, int total_tiles, int num_sms, cudaStream_t st) {
    static SmemAttrOnce once_p, once_t;
    int rc = ensure_smem_attr(reinterpret_cast<const void*>(xform_gemm_kernel<true>), (int)XG_SMEM, once_p);
    if (rc == SIE_OK) rc = ensure_smem_attr(reinterpret_cast<const void*>(xform_gemm_kernel<false>), (int)XG_SMEM, once_t);
    if (rc != SIE_OK) return rc;
    if (njobs <= 0 || total_tiles <= 0) return SIE_OK;
    const int grid = total_tiles < num_sms ? total_tiles : num_sms;
    if (packed)
        xform_gemm_kernel<true><<<grid, XG_THREADS, XG_SMEM, st>>>(d_jobs, njobs, total_tiles);
    else
        xform_gemm_kernel<false><<<grid, XG_THREADS, XG_SMEM, st>>>(d_jobs, njobs, total_tiles);
    note_launch();
    cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? SIE_OK : set_cuda_error(e);
}

// ------------------------------------------------------------------------------------------------
// grouped transposes: out[c][r] = in[r][c] for a list of (in, rows, cols, out, ld_out) jobs; blockIdx.z = job
__global__ void transpose_jobs_kernel(const TJob* __restrict__ jobs) {
    const TJob J = jobs[blockIdx.z];
    __shared__ double tile[32][33];
    const int r0 = blockIdx.y * 32, c0 = blockIdx.x * 32;
    if (r0 >= J.rows || c0 >= J.cols) return;
    for (int rr = threadIdx.y; rr < 32; rr += 8) {
        const int r = r0 + rr, c = c0 + threadIdx.x;
        tile[rr][threadIdx.x] = (r < J.rows && c < J.cols) ? J.in[(size_t)r * J.cols + c] : 0.0;
    }
    __syncthreads();
    for (int rr = threadIdx.y; rr < 32; rr += 8) {
        const int c = c0 + rr, r = r0 + threadIdx.x;
        if (c < J.cols && r < J.rows) J.out[(size_t)c * J.ld_out + r] = tile[threadIdx.x][rr];
    }
}
int launch_transpose_jobs(const TJob* d_jobs, int njobs, int max_rows, int max_cols, cudaStream_t st) {
    if (njobs <= 0) return SIE_OK;
    for (int z0 = 0; z0 < njobs; z0 += 65535) {
        const int nz = njobs - z0 < 65535 ? njobs - z0 : 65535;
        dim3 grid((max_cols + 31) / 32, (max_rows + 31) / 32, nz), block(32, 8);
        transpose_jobs_kernel<<<grid, block, 0, st>>>(d_jobs + z0);
        note_launch();
    }
    cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? SIE_OK : set_cuda_error(e);
}

// ------------------------------------------------------------------------------------------------
// Small device-side writers that keep descriptor and operand uploads OFF the host-to-device copy engine: that engine
// serves copies in order, so a 256-byte descriptor enqueued behind the 27.7 GB integral upload of the NEXT cluster
// (another plan, another stream) would hold this cluster's pair stage back for half a second.
struct PokeArgs {
    unsigned long long payload[64];  // up to 512 bytes, travels as a kernel parameter
    void* dst;
    int nwords;
};
__global__ void poke_kernel(const PokeArgs a) {
    unsigned long long* d = static_cast<unsigned long long*>(a.dst);
    for (int i = threadIdx.x; i < a.nwords; i += blockDim.x) d[i] = a.payload[i];
}
int launch_poke(const void* payload, size_t nbytes, void* dst, cudaStream_t st) {
    if (nbytes > 512 || (nbytes & 7)) return SIE_EINVAL;
    PokeArgs a;
    std::memcpy(a.payload, payload, nbytes);
    a.dst = dst;
    a.nwords = (int)(nbytes / 8);
    poke_kernel<<<1, 64, 0, st>>>(a);
    note_launch();
    cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? SIE_OK : set_cuda_error(e);
}
// dst[i] = src[i]; src may be pinned host memory mapped into the device address space (read over PCIe by the SMs)
__global__ void copy_f64_kernel(const double* __restrict__ src, double* __restrict__ dst, size_t n) {
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) dst[i] = src[i];
}
int launch_copy_f64(const double* src, double* dst, size_t n, cudaStream_t st) {
    if (n == 0) return SIE_OK;
    const int grid = (int)std::min<size_t>(64, (n + 255) / 256);
    copy_f64_kernel<<<grid, 256, 0, st>>>(src, dst, n);
    note_launch();
    cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? SIE_OK : set_cuda_error(e);
}

}  // namespace sie
