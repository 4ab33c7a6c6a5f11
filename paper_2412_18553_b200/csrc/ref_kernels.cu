// ref_kernels.cu — simple FP64-FMA CUDA kernels that follow the definition step by step in the "per-j" order of
// the problem statement.  Selected by SIE_FLAG_REFERENCE (and automatically for nocc > 128).  They exist as an
// on-device cross-check of the tensor-core path and as the any-size fallback; they are not tuned.
//   H^P_{i nu} = sum_mu C_{mu i} (P|mu nu);  B^P_{ia} = sum_nu H^P_{i nu} C_{nu a}          (Eq. S49)
//   for each j:  V^{ij}_{ab} = sum_P B^P_ia B^P_jb;   G[i'][i] += sum_ab V^{i'j}_ab / D * (2 V^{ij}_ab - V^{ij}_ba)
#include "sie_common.cuh"
#include "sie_internal.h"
#include "../../include/sie_dfmp2.h"

namespace sie {

// H[P][i][nu], thread per nu.
__global__ void ref_half1_kernel(const double* __restrict__ C_occ, const double* __restrict__ Lp, int nao, int o,
                                 double* __restrict__ H) {
    const int nu = blockIdx.x * blockDim.x + threadIdx.x, i = blockIdx.y, P = blockIdx.z;
    if (nu >= nao) return;
    const double* L = Lp + (size_t)P * ((size_t)nao * (nao + 1) / 2);
    double s = 0.0;
    for (int mu = 0; mu < nao; ++mu) {
        const size_t idx = mu >= nu ? (size_t)mu * (mu + 1) / 2 + nu : (size_t)nu * (nu + 1) / 2 + mu;
        s = fma(C_occ[(size_t)mu * o + i], L[idx], s);
    }
    H[((size_t)P * o + i) * nao + nu] = s;
}

// B[a][i][p0+P], thread per a.
__global__ void ref_half2_kernel(const double* __restrict__ H, const double* __restrict__ C_vir, int nao, int o, int v,
                                 int p0, double* __restrict__ B, int naux_ld) {
    const int a = blockIdx.x * blockDim.x + threadIdx.x, i = blockIdx.y, P = blockIdx.z;
    if (a >= v) return;
    const double* h = H + ((size_t)P * o + i) * nao;
    double s = 0.0;
    for (int nu = 0; nu < nao; ++nu) s = fma(h[nu], C_vir[(size_t)nu * v + a], s);
    B[((size_t)a * o + i) * naux_ld + p0 + P] = s;
}

int ref_transform(const double* C_occ, const double* C_vir, const double* Lp_block, int nao, int o, int v, int p0, int p1,
                  double* H, double* B, int naux_ld, cudaStream_t st) {
    const int np = p1 - p0;
    if (np <= 0) return SIE_OK;
    for (int z0 = 0; z0 < np; z0 += 32768) {
        const int nz = np - z0 < 32768 ? np - z0 : 32768;
        const double* Lz = Lp_block + (size_t)z0 * ((size_t)nao * (nao + 1) / 2);
        ref_half1_kernel<<<dim3((nao + 127) / 128, o, nz), 128, 0, st>>>(C_occ, Lz, nao, o, H);
        note_launch();
        ref_half2_kernel<<<dim3((v + 127) / 128, o, nz), 128, 0, st>>>(H, C_vir, nao, o, v, p0 + z0, B, naux_ld);
        note_launch();
    }
    cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? SIE_OK : set_cuda_error(e);
}

// Vj[i][a][b] = sum_P B[a][i][P] * B[b][j][P]; 16x16 outputs per CTA, K staged through shared memory.
__global__ void ref_vj_kernel(const double* __restrict__ B, int o, int v, int naux, int naux_ld, int j, double* __restrict__ Vj) {
    __shared__ double sa[16][17], sb[16][17];
    const int i = blockIdx.z;
    const int a = blockIdx.y * 16 + threadIdx.y, b = blockIdx.x * 16 + threadIdx.x;
    const int la = blockIdx.y * 16 + threadIdx.y, lb = blockIdx.x * 16 + threadIdx.y;  // rows loaded by this thread
    double s = 0.0;
    for (int k0 = 0; k0 < naux; k0 += 16) {
        const int k = k0 + threadIdx.x;
        sa[threadIdx.y][threadIdx.x] = (la < v && k < naux) ? B[((size_t)la * o + i) * naux_ld + k] : 0.0;
        sb[threadIdx.y][threadIdx.x] = (lb < v && k < naux) ? B[((size_t)lb * o + j) * naux_ld + k] : 0.0;
        __syncthreads();
#pragma unroll
        for (int kk = 0; kk < 16; ++kk) s = fma(sa[threadIdx.y][kk], sb[threadIdx.x][kk], s);
        __syncthreads();
    }
    if (a < v && b < v) Vj[((size_t)i * v + a) * v + b] = s;
}

// G[i'][i] += sum_ab Vj[i'][a][b] / (e_i' + e_j - e_a - e_b) * (2 Vj[i][a][b] - Vj[i][b][a]); one CTA per (i', i).
__global__ void __launch_bounds__(256) ref_g_kernel(const double* __restrict__ Vj, int o, int v, int j,
                                                    const double* __restrict__ e_occ, const double* __restrict__ e_vir,
                                                    double* __restrict__ G, int mode) {
    const int ip = blockIdx.y, i = blockIdx.x;
    const double* Vp = Vj + (size_t)ip * v * v;
    const double* Vi = Vj + (size_t)i * v * v;
    const double eij = e_occ[ip] + e_occ[j];
    double s = 0.0;
    for (int ab = threadIdx.x; ab < v * v; ab += 256) {
        const int a = ab / v, b = ab - a * v;
        const double D = (eij - e_vir[a]) - e_vir[b];
        const double w = 2.0 * Vi[ab] - Vi[(size_t)b * v + a];
        // mode 1 (Eq. S18): the second factor is an amplitude too, t_{ij}^{ab} and t_{ij}^{ba} share D_{ij}^{ab}
        s = fma(Vp[ab] / D, mode ? w / (((e_occ[i] + e_occ[j]) - e_vir[a]) - e_vir[b]) : w, s);
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
    __shared__ double ws[8];
    if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double tot = 0.0;
        for (int w = 0; w < 8; ++w) tot += ws[w];
        G[(size_t)ip * o + i] += tot;
    }
}

size_t ref_vj_bytes(int o, int v) { return (size_t)o * v * v * sizeof(double); }

int ref_pair(const double* B, int o, int v, int naux, int naux_ld, const double* e_occ, const double* e_vir, double* Vj,
             double* G, int mode, cudaStream_t st) {
    cudaError_t e = cudaMemsetAsync(G, 0, (size_t)o * o * sizeof(double), st);
    if (e != cudaSuccess) return set_cuda_error(e);
    for (int j = 0; j < o; ++j) {
        ref_vj_kernel<<<dim3((v + 15) / 16, (v + 15) / 16, o), dim3(16, 16), 0, st>>>(B, o, v, naux, naux_ld, j, Vj);
        note_launch();
        ref_g_kernel<<<dim3(o, o), 256, 0, st>>>(Vj, o, v, j, e_occ, e_vir, G, mode);
        note_launch();
    }
    e = cudaGetLastError();
    return e == cudaSuccess ? SIE_OK : set_cuda_error(e);
}

}  // namespace sie
