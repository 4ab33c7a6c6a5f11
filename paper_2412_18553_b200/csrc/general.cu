// general.cu — the any-size pair stage: G (energy path), gamma_occ (Eq. S18) and gamma_vir (Eq. S17) for orbital sets the fused
// kernel does not cover (nocc > 128: the environment-occupied sub-space of PAPER.md Eq. S13) and for gamma_vir
// at every size.  Same mathematics as pair.cu, organised as three grouped launches per occupied block K = [k0, k0+Kb):
//
//   1. slab GEMM      V[(a,i)][(b,k)] = sum_P B[a][i][P] B[b][k][P]     all (a,i), all b, k in K    (xform_gemm_kernel, TMA both sides)
//   2. combine        S1 = V / D,  S2 = 2V - V~ (G)  or  (2V - V~) / D (gamma),   V~ = V[(b,i)][(a,k)] = (ib|ka),
//                     D = e_i + e_k - e_a - e_b                                          Eq. S15-S16 (L348-L351)
//   3. Gram GEMM      G[i'][i]      += sum_{a,b,k} S1[i'][(a,b,k)] S2[i][(a,b,k)]        energy path / Eq. S18 (L357)
//                     gamma_vir[a][c] += sum_{i,b,k} S1[a][(i,b,k)] S2[c][(i,b,k)]       Eq. S17 (L355), b the summed virtual
//      split over K-ranges into partial slots that reduce_trace_kernel sums in fixed order (no atomics).
//
// Block-slab mode: the amplitude slab of one occupied block (<= 1 GB, power-of-two block) is the only O(n^4)-shaped object
// and it lives for one block; the slab GEMM forms ordered pairs (i,k), i.e. twice the SYRK minimum of the fused kernel.
// Whole-matrix mode (general_geom().full: the integral matrix (o v)^2 doubles fits in 8 GB — the large-occ x small-vir
// sub-space of the BNO step and every small cluster): one block covers the cluster and stage 1 is a SYRK (one job per
// 128-row block from its diagonal on, lower triangle mirrored): the o^2 v^2 naux minimum.
#include <algorithm>
#include <cstring>
#include <vector>

#include "sie_common.cuh"
#include "sie_internal.h"
#include "../../include/sie_dfmp2.h"

namespace sie {

// mode 0: S1 = t, S2 = 2V - V~        rows of S: i, columns (a, col)      -> G[i'][i]
// mode 1: S1 = t, S2 = 2t - t~        rows of S: i, columns (a, col)      -> Gamma_occ
// mode 2: S1 = t, S2 = 2t - t~        rows of S: a, columns (i, col)      -> gamma_vir / 2
// col = b * Kb + kl (kl the index inside the occupied block), ldc = ceil8(v * Kb); padding columns and k >= o are written 0.
__global__ void slab_combine_kernel(const double* __restrict__ V, int o, int v, int Kb, int k0, int ldc, const double* __restrict__ e_occ,
                                    const double* __restrict__ e_vir, int mode, double* __restrict__ S1, double* __restrict__ S2) {
    const long long total = (long long)v * o * ldc;
    for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < total; e += (long long)gridDim.x * blockDim.x) {
        const int col = (int)(e % ldc);
        const long long row = e / ldc;  // a * o + i
        const int a = (int)(row / o), i = (int)(row - (long long)a * o);
        const int b = col / Kb, kl = col - b * Kb, k = k0 + kl;
        double s1 = 0.0, s2 = 0.0;
        if (b < v && k < o) {
            const double x = V[e];
            const double y = V[((long long)b * o + i) * ldc + a * Kb + kl];  // (ib|ka)
            const double D = ((e_occ[i] + e_occ[k]) - e_vir[a]) - e_vir[b];
            s1 = x / D;
            s2 = mode == 0 ? fma(2.0, x, -y) : fma(2.0, x, -y) / D;
        }
        const long long dst = mode == 2 ? e : ((long long)i * v + a) * ldc + col;
        S1[dst] = s1;
        S2[dst] = s2;
    }
}

// V[r][c] = V[c][r] for r > c (square n x n, leading dimension ld): completes a matrix whose upper triangle was computed
__global__ void mirror_lower_kernel(double* __restrict__ V, long long n, long long ld) {
    __shared__ double tile[32][33];
    const long long bc = blockIdx.x, br = blockIdx.y;  // destination tile (rows br, columns bc), only br >= bc
    if (br < bc) return;
    for (int rr = threadIdx.y; rr < 32; rr += 8) {  // read the source tile (rows bc-block, columns br-block), coalesced
        const long long r = bc * 32 + rr, c = br * 32 + threadIdx.x;
        tile[rr][threadIdx.x] = (r < n && c < n) ? V[r * ld + c] : 0.0;
    }
    __syncthreads();
    for (int rr = threadIdx.y; rr < 32; rr += 8) {
        const long long r = br * 32 + rr, c = bc * 32 + threadIdx.x;
        if (r < n && c < n && r > c) V[r * ld + c] = tile[threadIdx.x][rr];
    }
}

int launch_mirror_lower(double* V, long long n, long long ld, cudaStream_t st) {
    const unsigned nb32 = (unsigned)((n + 31) / 32);
    mirror_lower_kernel<<<dim3(nb32, nb32), dim3(32, 8), 0, st>>>(V, n, ld);
    note_launch();
    cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? SIE_OK : set_cuda_error(e);
}

GeneralGeom general_geom(int o, int v, int num_sms) {
    GeneralGeom g{};
    int Kb = 1;
    while (Kb * 2 <= std::min(o, 128) && (double)v * o * v * (Kb * 2) * 8.0 <= (double)((size_t)1 << 30)) Kb *= 2;
    // When the whole integral matrix M[(a,i)][(b,k)] = (ia|kb) fits (<= 8 GB: the large-occ x small-vir sub-space of the BNO
    // step, and every small cluster), ONE occupied block covers everything and the slab GEMM becomes a SYRK: only the tile
    // rows' upper parts are computed and the lower triangle is mirrored — the o^2 v^2 naux minimum instead of twice that.
    g.full = (double)v * o * (double)v * o * 8.0 <= 8.0 * (double)((size_t)1 << 30);
    if (g.full) Kb = o;
    g.Kb = Kb;
    g.ldc = (int)align_up((size_t)v * Kb, 8);
    g.slab_bytes = align_up((size_t)v * o * g.ldc * 8, 256);
    g.ok = (double)g.slab_bytes <= (double)((size_t)(g.full ? 9 : 4) << 30);
    for (int which = 0; which < 2; ++which) {  // Gram of the occupied (0) / virtual (1) block: split K until ~4 waves of tiles
        const int n = which ? v : o;
        const int mt = (n + 127) / 128, tiles = mt * ((n + 127) / 128);
        int ns = (4 * num_sms + tiles - 1) / tiles;
        ns = std::max(1, std::min(ns, 64));
        (which ? g.nsplit_vir : g.nsplit_occ) = ns;
    }
    g.slots_bytes = align_up(std::max((size_t)g.nsplit_occ * o * o, (size_t)g.nsplit_vir * v * v) * 8, 256);
    g.max_jobs = 1 + std::max(g.nsplit_occ, g.nsplit_vir);
    if (g.full) g.max_jobs += (int)(((long long)v * o + 127) / 128);  // one SYRK job per 128-row block
    return g;
}

// Runs the three stages for every occupied block and leaves the partial results in `slots` ([nsplit][n*n], n = o or v).
// scratch: 3 slabs (V, S1, S2) + job arena of (1 + nsplit) XJobs per occupied block.
int general_pair(const GeneralGeom& g, const double* Bmat, int o, int v, int naux, int naux_ld, const double* e_occ, const double* e_vir,
                 int mode, unsigned char* scratch, double* slots, int* nslots, int num_sms, cudaStream_t st) {
    const int n = mode == 2 ? v : o, nsplit = mode == 2 ? g.nsplit_vir : g.nsplit_occ;
    double* V = reinterpret_cast<double*>(scratch);
    double* S1 = reinterpret_cast<double*>(scratch + g.slab_bytes);
    double* S2 = reinterpret_cast<double*>(scratch + 2 * g.slab_bytes);
    unsigned char* arena = scratch + 3 * g.slab_bytes;
    const int nblocks = (o + g.Kb - 1) / g.Kb;
    cudaError_t ce = cudaMemsetAsync(slots, 0, (size_t)nsplit * n * n * 8, st);
    if (ce != cudaSuccess) return set_cuda_error(ce);
    const long long rows = (long long)v * o;
    std::vector<XJob> jobs;
    for (int blk = 0; blk < nblocks; ++blk) {
        const int k0 = blk * g.Kb;
        unsigned char* d_jobs = arena + (size_t)blk * g.max_jobs * sizeof(XJob);
        // ---- 1. slab GEMM
        int first_gram_job = 1;
        if (g.full) {
            // SYRK of the (v*o) x naux matrix B: one job per 128-row block r, columns from r*128 on; then mirror
            jobs.clear();
            const int nrb = (int)((rows + 127) / 128);
            long long t = 0;
            for (int r = 0; r < nrb; ++r) {
                const long long r0 = (long long)r * 128, M = std::min<long long>(128, rows - r0), N = rows - r0;
                XJob J;
                std::memset(&J, 0, sizeof J);
                const double* Br = Bmat + r0 * naux_ld;
                int rc = make_tensor_map_3d(&J.mapA, Br, naux, M, 1, (uint64_t)naux_ld * 8, (uint64_t)M * naux_ld * 8, 8, (uint32_t)(8 * ((M + 7) / 8)), 1);
                if (rc != SIE_OK) return rc;
                rc = make_tensor_map_3d(&J.mapB, Br, naux, N, 1, (uint64_t)naux_ld * 8, (uint64_t)N * naux_ld * 8, 8, 128, 1);
                if (rc != SIE_OK) return rc;
                J.n_total = N;
                J.M = (int)M;
                J.m8 = (int)((M + 7) / 8);
                J.m_tiles = 1;
                J.n_tiles = (int)((N + 127) / 128);
                J.kblocks = (naux + 7) / 8;
                J.b_c1_mul = 128;
                J.out.base = V + r0 * g.ldc + r0;
                J.out.ld_m = g.ldc;
                J.out.M = (int)M;
                J.out.inner = g.ldc;
                J.out.valid_inner = (int)N;
                J.out.stride_outer = 0;
                J.out.n_lin_total = N;
                J.tile_begin = (int)t;
                t += J.n_tiles;
                jobs.push_back(J);
            }
            ce = cudaMemcpyAsync(d_jobs, jobs.data(), jobs.size() * sizeof(XJob), cudaMemcpyHostToDevice, st);
            if (ce != cudaSuccess) return set_cuda_error(ce);
            int rc = launch_xform_gemm(false, reinterpret_cast<const XJob*>(d_jobs), (int)jobs.size(), (int)t, num_sms, st);
            if (rc != SIE_OK) return rc;
            const unsigned nb32 = (unsigned)((rows + 31) / 32);
            mirror_lower_kernel<<<dim3(nb32, nb32), dim3(32, 8), 0, st>>>(V, rows, g.ldc);
            note_launch();
            ce = cudaGetLastError();
            if (ce != cudaSuccess) return set_cuda_error(ce);
            first_gram_job = (int)jobs.size();
        } else {
        XJob J;
        std::memset(&J, 0, sizeof J);
        int rc = make_tensor_map_3d(&J.mapA, Bmat, naux, rows, 1, (uint64_t)naux_ld * 8, (uint64_t)rows * naux_ld * 8, 8, 128, 1);
        if (rc != SIE_OK) return rc;
        rc = make_tensor_map_3d(&J.mapB, Bmat, naux, o, v, (uint64_t)naux_ld * 8, (uint64_t)o * naux_ld * 8, 8, g.Kb, 128 / g.Kb);
        if (rc != SIE_OK) return rc;
        J.n_total = (long long)v * g.Kb;
        J.M = (int)rows;
        J.m8 = 16;
        J.m_tiles = (int)((rows + 127) / 128);
        J.n_tiles = (int)((J.n_total + 127) / 128);
        J.kblocks = (naux + 7) / 8;
        J.b_c1_off = k0;
        J.b_c1_mul = 0;
        J.b_c2_mul = 128 / g.Kb;
        J.out.base = V;
        J.out.ld_m = g.ldc;
        J.out.M = (int)rows;
        J.out.inner = g.ldc;
        J.out.valid_inner = v * g.Kb;
        J.out.stride_outer = 0;
        J.out.n_lin_total = J.n_total;
        J.tile_begin = 0;
        ce = cudaMemcpyAsync(d_jobs, &J, sizeof J, cudaMemcpyHostToDevice, st);
        if (ce != cudaSuccess) return set_cuda_error(ce);
        rc = launch_xform_gemm(false, reinterpret_cast<const XJob*>(d_jobs), 1, J.m_tiles * J.n_tiles, num_sms, st);
        if (rc != SIE_OK) return rc;
        }
        // ---- 2. amplitudes and the 2x - x~ combination
        slab_combine_kernel<<<num_sms * 8, 256, 0, st>>>(V, o, v, g.Kb, k0, g.ldc, e_occ, e_vir, mode, S1, S2);
        note_launch();
        ce = cudaGetLastError();
        if (ce != cudaSuccess) return set_cuda_error(ce);
        // ---- 3. Gram GEMM, split over K into the partial slots
        const long long Ktot = (long long)(mode == 2 ? o : v) * g.ldc;  // multiple of 8
        const int kblocks = (int)(Ktot / 8);
        int kchunk = (kblocks + nsplit - 1) / nsplit;
        kchunk = (kchunk + 1) / 2 * 2;  // two K-blocks per pipeline stage: ranges must not share a stage
        jobs.clear();
        int t = 0;
        for (int s = 0; s < nsplit; ++s) {
            const int kb0 = s * kchunk;
            if (kb0 >= kblocks) break;
            XJob Q;
            std::memset(&Q, 0, sizeof Q);
            const int mt = (n + 127) / 128, m8 = ((n + mt - 1) / mt + 7) / 8;
            int rc = make_tensor_map_3d(&Q.mapA, S1, (uint64_t)Ktot, n, 1, (uint64_t)Ktot * 8, (uint64_t)Ktot * 8 * n, 8, 8 * m8, 1);
            if (rc != SIE_OK) return rc;
            rc = make_tensor_map_3d(&Q.mapB, S2, (uint64_t)Ktot, n, 1, (uint64_t)Ktot * 8, (uint64_t)Ktot * 8 * n, 8, 128, 1);
            if (rc != SIE_OK) return rc;
            Q.n_total = n;
            Q.M = n;
            Q.m8 = m8;
            Q.m_tiles = (n + 8 * m8 - 1) / (8 * m8);
            Q.n_tiles = (n + 127) / 128;
            Q.kblocks = std::min(kchunk, kblocks - kb0);
            Q.k0_blocks = kb0;
            Q.b_c1_mul = 128;
            Q.out.base = slots + (size_t)s * n * n;
            Q.out.ld_m = n;
            Q.out.M = n;
            Q.out.inner = n;
            Q.out.valid_inner = n;
            Q.out.stride_outer = 0;
            Q.out.n_lin_total = n;
            Q.out.accumulate = 1;
            Q.tile_begin = t;
            t += Q.m_tiles * Q.n_tiles;
            jobs.push_back(Q);
        }
        ce = cudaMemcpyAsync(d_jobs + (size_t)first_gram_job * sizeof(XJob), jobs.data(), jobs.size() * sizeof(XJob), cudaMemcpyHostToDevice, st);
        if (ce != cudaSuccess) return set_cuda_error(ce);
        int rc = launch_xform_gemm(false, reinterpret_cast<const XJob*>(d_jobs + (size_t)first_gram_job * sizeof(XJob)), (int)jobs.size(), t,
                                   num_sms, st);
        if (rc != SIE_OK) return rc;
    }
    *nslots = nsplit;
    return SIE_OK;
}

size_t general_scratch_bytes(const GeneralGeom& g, int o) {
    const int nblocks = (o + g.Kb - 1) / g.Kb;
    return 3 * g.slab_bytes + align_up((size_t)nblocks * g.max_jobs * sizeof(XJob), 256);
}

}  // namespace sie
