// canonical.cu — NEXT-2: closed-shell canonical DF-MP2 correlation energy of a WHOLE system,
//     E_MP2 = sum_{ij} sum_{ab} (ia|jb) ( 2 (ia|jb) - (ib|ja) ) / (e_i + e_j - e_a - e_b)        (Eq. S15-S16, P_frag = I)
// the E_MP2 term of the bath-truncation correction (PAPER.md Eq. S63; Eq. S68) and the paper's only timed
// MP2 (Table S1).  At N ~ 6k-11k orbitals B^P_ia (o * v * naux doubles) no longer fits in device memory, so:
//
//   phase 1 (sie_dfmp2_canonical_transform)  aux rows [p0,p1) -> B[i][a][P] written into a B STORE the caller owns
//       (pinned host memory for the out-of-core case, device memory when it fits — any pointer cudaMemcpy understands);
//       same grouped A1/A2 tensor-core GEMMs as the cluster path, A1 fed from the packed integrals.
//   phase 2 (sie_dfmp2_canonical_energy)     occupied-block pairs I <= K: panels B_I, B_K are brought to the device
//       (double-buffered copy stream), one GEMM forms V[(i,a)][(k,b)] for the whole block pair (unordered occupied pairs:
//       the o^2 v^2 naux minimum), and an elementwise pass adds w * V (2V - V~) / D into CTA-private slots
//       (w = 2 for I < K); the slots are summed in fixed order.  V lives for one block pair; amplitudes are never stored.
#include <algorithm>
#include <cstring>
#include <new>
#include <vector>

#include "../../include/sie_dfmp2.h"
#include "sie_common.cuh"
#include "sie_internal.h"

namespace sie {

constexpr int CAN_GRID = 1184;  // 148 x 8 CTAs of the energy pass, each with a private partial-sum slot

// V [(i,a)][(k,b)] with leading dimension ldv; rows i in [0,ni), columns k in [0,nk); e_i / e_k point at the blocks' energies.
// The exchange partner (ib|ka) of an element is its transpose INSIDE the v x v block of one (i,k) pair, so the block is walked
// in pairs of 32 x 32 tiles (ta <= tb): both tiles are read once with coalesced rows, the transposed operand comes from
// shared memory, and one tile pair yields the terms of (a,b) and of (b,a) — V is read from HBM exactly once (an
// element-wise walk fetched a 32-byte sector for every 8-byte partner: 4.5x the bytes).
__global__ void __launch_bounds__(256) canonical_energy_kernel(const double* __restrict__ V, int ni, int nk, int v, long long ldv,
                                                                const double* __restrict__ e_i, const double* __restrict__ e_k,
                                                                const double* __restrict__ e_vir, double weight, double* __restrict__ slots) {
    __shared__ double T1[32][33], T2[32][33];
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const int nt = (v + 31) / 32;
    const long long ntp = (long long)nt * (nt + 1) / 2, total = (long long)ni * nk * ntp;
    double s = 0.0;
    for (long long item = blockIdx.x; item < total; item += gridDim.x) {
        const long long ik = item / ntp;
        int rem = (int)(item - ik * ntp), ta = 0;
        while (rem >= nt - ta) {
            rem -= nt - ta;
            ++ta;
        }
        const int tb = ta + rem;
        const int i = (int)(ik / nk), k = (int)(ik - (long long)i * nk);
        const int a0 = 32 * ta, b0 = 32 * tb;
        const double* blk = V + (long long)i * v * ldv + (long long)k * v;  // V_ik [a][b], row stride ldv
#pragma unroll
        for (int r = ty; r < 32; r += 8) {
            const bool in1 = a0 + r < v && b0 + tx < v, in2 = b0 + r < v && a0 + tx < v;
            T1[r][tx] = in1 ? blk[(long long)(a0 + r) * ldv + b0 + tx] : 0.0;
            T2[r][tx] = (ta != tb && in2) ? blk[(long long)(b0 + r) * ldv + a0 + tx] : 0.0;
        }
        __syncthreads();
        const double eik = e_i[i] + e_k[k];
        const int b = b0 + tx;
        if (b < v) {
            const double eb = e_vir[b];
#pragma unroll
            for (int r = ty; r < 32; r += 8) {
                const int a = a0 + r;
                if (a >= v) break;
                const double D = (eik - e_vir[a]) - eb;
                const double x = T1[r][tx];
                if (ta == tb) {
                    const double y = T1[tx][r];  // (ib|ka) of the same tile
                    s += x * fma(2.0, x, -y) / D;
                } else {
                    const double y = T2[tx][r];  // element (b,a) of the block: the (a,b) term and the (b,a) term share D
                    s += (x * fma(2.0, x, -y) + y * fma(2.0, y, -x)) / D;
                }
            }
        }
        __syncthreads();
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
    __shared__ double wsum[8];
    if ((threadIdx.x & 31) == 0) wsum[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
#pragma unroll
        for (int w = 0; w < 8; ++w) t += wsum[w];
        slots[blockIdx.x] += weight * t;  // CTA-private slot, launches are stream-ordered: fixed summation order
    }
}

}  // namespace sie

using namespace sie;

struct sie_dfmp2_canon_s {
    int nao = 0, o = 0, v = 0, naux = 0, nao_ld = 0, naux_ld = 0, pblk = 0, pbld = 0, Ib = 0, num_sms = 148;
    size_t npair = 0;
    size_t off_CoT = 0, off_CvT = 0, off_H = 0, off_Bblk = 0, off_jobs = 0, off_panel = 0, off_V = 0, off_slots = 0, off_rc = 0, total = 0;
    size_t panel_bytes = 0;
    long long ldv = 0;
    int max_jobs = 0;
    bool coeffs_ready = false;
    const void* ws_ready = nullptr;
    long long covered_rows = 0;
    std::vector<std::pair<int, int>> covered;
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t ev_ready[2] = {nullptr, nullptr}, ev_free[2] = {nullptr, nullptr}, ev_fork = nullptr;
};

namespace {

#define CAN_CUDA(call)                                        \
    do {                                                      \
        cudaError_t e__ = (call);                             \
        if (e__ != cudaSuccess) return set_cuda_error(e__);   \
    } while (0)
#define CAN_TRY(call)                     \
    do {                                  \
        int rc__ = (call);                \
        if (rc__ != SIE_OK) return rc__;  \
    } while (0)

struct Carve {
    size_t off = 0;
    size_t take(size_t bytes) {
        size_t r = off;
        off = align_up(off + bytes, 256);
        return r;
    }
};

// plain K-major GEMM job C[m][n] = sum_k A[m][k] Bop[n][k] with M rows cut into near-equal chunks of at most 128
int gemm_job(XJob& J, const double* A, long long M, const double* Bop, long long N, int K, int ld, const GemmOut& out) {
    std::memset(&J, 0, sizeof J);
    const int m_tiles = (int)((M + 127) / 128);
    const int m8 = (int)(((M + m_tiles - 1) / m_tiles + 7) / 8);
    CAN_TRY(make_tensor_map_3d(&J.mapA, A, K, M, 1, (uint64_t)ld * 8, (uint64_t)ld * 8 * M, 8, 8 * m8, 1));
    CAN_TRY(make_tensor_map_3d(&J.mapB, Bop, K, N, 1, (uint64_t)ld * 8, (uint64_t)ld * 8 * N, 8, 128, 1));
    J.n_total = N;
    J.M = (int)M;
    J.m8 = m8;
    J.m_tiles = (int)((M + 8 * m8 - 1) / (8 * m8));
    J.n_tiles = (int)((N + 127) / 128);
    J.kblocks = (K + 7) / 8;
    J.b_c1_mul = 128;
    J.out = out;
    return SIE_OK;
}

int ensure_streams(sie_dfmp2_canon_s& p) {
    if (p.copy_stream) return SIE_OK;
    CAN_CUDA(cudaStreamCreateWithFlags(&p.copy_stream, cudaStreamNonBlocking));
    for (int i = 0; i < 2; ++i) {
        CAN_CUDA(cudaEventCreateWithFlags(&p.ev_ready[i], cudaEventDisableTiming));
        CAN_CUDA(cudaEventCreateWithFlags(&p.ev_free[i], cudaEventDisableTiming));
    }
    CAN_CUDA(cudaEventCreateWithFlags(&p.ev_fork, cudaEventDisableTiming));
    return SIE_OK;
}

}  // namespace

extern "C" {

int sie_dfmp2_canonical_plan(sie_dfmp2_canon_t* plan, int nao, int nocc, int nvir, int naux, int occ_block, size_t* workspace_bytes,
                             size_t* bstore_bytes) {
    if (!plan || !workspace_bytes || !bstore_bytes) return SIE_EINVAL;
    if (nao < 1 || nocc < 1 || nvir < 1 || naux < 1 || occ_block < 0 || (long long)nocc + nvir > nao) return SIE_EINVAL;
    sie_dfmp2_canon_s* p = new (std::nothrow) sie_dfmp2_canon_s();
    if (!p) return SIE_ENOMEM;
    p->nao = nao, p->o = nocc, p->v = nvir, p->naux = naux;
    p->nao_ld = (int)align_up((size_t)nao, 8);
    p->naux_ld = (int)align_up((size_t)naux, 8);
    p->npair = (size_t)nao * (nao + 1) / 2;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && sms > 0)
        p->num_sms = sms;
    else
        (void)cudaGetLastError();
    // aux sub-block of the transform: H <= 1 GB, the B block buffer <= 2 GB, flat GEMM column indices below 2^31
    long long pb = std::min<long long>((long long)(((size_t)1 << 30) / ((size_t)nocc * p->nao_ld * 8)),
                                       (long long)(((size_t)2 << 30) / ((size_t)nocc * nvir * 8)));
    pb = std::min<long long>(pb, (long long)0x7fffffff / std::max(nao, nocc) - 1);
    pb = std::max<long long>(8, pb / 8 * 8);
    p->pblk = (int)std::min<long long>(pb, naux);
    p->pbld = (int)align_up((size_t)p->pblk, 8);
    // occupied block of the pair phase: three panels [Ib][v][naux_ld] and V [(Ib v)][(Ib v)] within ~12 GB
    int Ib = occ_block > 0 ? std::min(occ_block, nocc) : nocc;
    if (occ_block == 0) {
        const double budget = 12.0 * (double)((size_t)1 << 30);
        while (Ib > 1 && 3.0 * Ib * nvir * p->naux_ld * 8.0 + (double)Ib * nvir * (double)Ib * nvir * 8.0 > budget) Ib = (Ib + 1) / 2;
    }
    if ((long long)Ib * nvir > 0x3fffffff) {
        delete p;
        return SIE_EINVAL;
    }
    p->Ib = Ib;
    p->ldv = (long long)align_up((size_t)Ib * nvir, 8);
    p->panel_bytes = align_up((size_t)Ib * nvir * p->naux_ld * 8, 256);
    p->max_jobs = 4 + (int)(((long long)Ib * nvir + 127) / 128);  // + one SYRK job per 128-row block of a diagonal block pair
    Carve c;
    p->off_CoT = c.take((size_t)nocc * p->nao_ld * 8);
    p->off_CvT = c.take((size_t)nvir * p->nao_ld * 8);
    p->off_H = c.take((size_t)nocc * p->pblk * p->nao_ld * 8);
    p->off_Bblk = c.take((size_t)nocc * nvir * p->pbld * 8);
    p->off_jobs = c.take((size_t)p->max_jobs * sizeof(XJob) + 2 * sizeof(TJob));
    p->off_panel = c.take(3 * p->panel_bytes);
    p->off_V = c.take((size_t)Ib * nvir * p->ldv * 8);
    p->off_slots = c.take((size_t)CAN_GRID * 8);
    p->off_rc = c.take(sizeof(ReduceCluster));
    p->total = c.off;
    *plan = p;
    *workspace_bytes = p->total;
    *bstore_bytes = (size_t)nocc * nvir * p->naux_ld * 8;
    return SIE_OK;
}

int sie_dfmp2_canonical_transform(sie_dfmp2_canon_t plan, void* workspace, const double* C_occ, const double* C_vir,
                                  const double* L_packed_block, int p0, int p1, double* B_store, void* cuda_stream) {
    if (!plan || !workspace || !C_occ || !C_vir || !L_packed_block || !B_store) return SIE_EINVAL;
    sie_dfmp2_canon_s& p = *plan;
    if (p0 < 0 || p1 > p.naux || p0 >= p1 || (reinterpret_cast<uintptr_t>(workspace) & 255)) return SIE_EINVAL;
    if (!p.covered.empty() && p.ws_ready != workspace) return SIE_ESTATE;
    for (auto& iv : p.covered)
        if (p0 < iv.second && iv.first < p1) return SIE_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    unsigned char* ws = static_cast<unsigned char*>(workspace);
    double* CoT = reinterpret_cast<double*>(ws + p.off_CoT);
    double* CvT = reinterpret_cast<double*>(ws + p.off_CvT);
    double* H = reinterpret_cast<double*>(ws + p.off_H);
    double* Bblk = reinterpret_cast<double*>(ws + p.off_Bblk);
    unsigned char* arena = ws + p.off_jobs;
    if (p.ws_ready != workspace) {
        TJob tj[2] = {{C_occ, CoT, p.nao, p.o, p.nao_ld, 0}, {C_vir, CvT, p.nao, p.v, p.nao_ld, 0}};
        unsigned char* d = arena + (size_t)p.max_jobs * sizeof(XJob);
        CAN_CUDA(cudaMemcpyAsync(d, tj, sizeof tj, cudaMemcpyHostToDevice, st));
        CAN_TRY(launch_transpose_jobs(reinterpret_cast<const TJob*>(d), 2, p.nao, std::max(p.o, p.v), st));
        p.ws_ready = workspace;
    }
    for (int q0 = p0; q0 < p1; q0 += p.pblk) {
        const int q1 = std::min(p1, q0 + p.pblk), pb = q1 - q0;
        // A1: H[i][P][nu] from the packed rows (gathered by the producer warps, see transform.cu)
        XJob J;
        GemmOut o1{};
        o1.base = H, o1.ld_m = (long long)pb * p.nao_ld, o1.M = p.o, o1.inner = p.nao, o1.valid_inner = p.nao, o1.stride_outer = p.nao_ld;
        o1.n_lin_total = (long long)pb * p.nao;
        CAN_TRY(gemm_job(J, CoT, p.o, CoT /*unused in packed mode*/, 128, p.nao, p.nao_ld, o1));
        J.Lp = L_packed_block + (size_t)(q0 - p0) * p.npair;
        J.npair = (long long)p.npair;
        J.nao = p.nao;
        J.n_total = (long long)pb * p.nao;
        J.n_tiles = (int)((J.n_total + 127) / 128);
        CAN_CUDA(cudaMemcpyAsync(arena, &J, sizeof J, cudaMemcpyHostToDevice, st));
        CAN_TRY(launch_xform_gemm(true, reinterpret_cast<const XJob*>(arena), 1, J.m_tiles * J.n_tiles, p.num_sms, st));
        // A2: Bblk[i][a][P] (occupied-major, aux contiguous) = sum_nu CvT[a][nu] H[(i,P)][nu]
        GemmOut o2{};
        o2.base = Bblk, o2.ld_m = p.pbld, o2.M = p.v, o2.inner = pb, o2.valid_inner = pb, o2.stride_outer = (long long)p.v * p.pbld;
        o2.n_lin_total = (long long)p.o * pb;
        CAN_TRY(gemm_job(J, CvT, p.v, H, (long long)p.o * pb, p.nao, p.nao_ld, o2));
        CAN_CUDA(cudaMemcpyAsync(arena + sizeof(XJob), &J, sizeof J, cudaMemcpyHostToDevice, st));
        CAN_TRY(launch_xform_gemm(false, reinterpret_cast<const XJob*>(arena + sizeof(XJob)), 1, J.m_tiles * J.n_tiles, p.num_sms, st));
        // into the store: rows (i,a) of naux_ld doubles, columns [q0, q1)
        CAN_CUDA(cudaMemcpy2DAsync(B_store + q0, (size_t)p.naux_ld * 8, Bblk, (size_t)p.pbld * 8, (size_t)pb * 8, (size_t)p.o * p.v,
                                   cudaMemcpyDefault, st));
    }
    p.covered.emplace_back(p0, p1);
    p.covered_rows += p1 - p0;
    return SIE_OK;
}

int sie_dfmp2_canonical_energy(sie_dfmp2_canon_t plan, void* workspace, const double* e_occ, const double* e_vir, const double* B_store,
                               double* E_out, void* cuda_stream) {
    if (!plan || !workspace || !e_occ || !e_vir || !B_store || !E_out) return SIE_EINVAL;
    sie_dfmp2_canon_s& p = *plan;
    if (p.covered_rows != p.naux) return SIE_ESTATE;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    unsigned char* ws = static_cast<unsigned char*>(workspace);
    double* panel[3] = {reinterpret_cast<double*>(ws + p.off_panel), reinterpret_cast<double*>(ws + p.off_panel + p.panel_bytes),
                        reinterpret_cast<double*>(ws + p.off_panel + 2 * p.panel_bytes)};
    double* V = reinterpret_cast<double*>(ws + p.off_V);
    double* slots = reinterpret_cast<double*>(ws + p.off_slots);
    unsigned char* arena = ws + p.off_jobs;
    CAN_TRY(ensure_streams(p));
    CAN_CUDA(cudaMemsetAsync(slots, 0, (size_t)CAN_GRID * 8, st));
    CAN_CUDA(cudaEventRecord(p.ev_fork, st));
    CAN_CUDA(cudaStreamWaitEvent(p.copy_stream, p.ev_fork, 0));
    const int nblk = (p.o + p.Ib - 1) / p.Ib;
    const size_t row_doubles = (size_t)p.v * p.naux_ld;  // one occupied orbital of the store
    int turn = 0;
    for (int I = 0; I < nblk; ++I) {
        const int i0 = I * p.Ib, ni = std::min(p.Ib, p.o - i0);
        CAN_CUDA(cudaMemcpyAsync(panel[0], B_store + (size_t)i0 * row_doubles, (size_t)ni * row_doubles * 8, cudaMemcpyDefault, st));
        for (int K = I; K < nblk; ++K) {
            const int k0 = K * p.Ib, nk = std::min(p.Ib, p.o - k0);
            const double* PK = panel[0];
            int buf = -1;
            if (K != I) {  // panel of block K through the two-buffer ring on the copy stream, under the GEMM of the pair before
                buf = turn++ & 1;
                CAN_CUDA(cudaStreamWaitEvent(p.copy_stream, p.ev_free[buf], 0));
                CAN_CUDA(cudaMemcpyAsync(panel[1 + buf], B_store + (size_t)k0 * row_doubles, (size_t)nk * row_doubles * 8, cudaMemcpyDefault,
                                         p.copy_stream));
                CAN_CUDA(cudaEventRecord(p.ev_ready[buf], p.copy_stream));
                CAN_CUDA(cudaStreamWaitEvent(st, p.ev_ready[buf], 0));
                PK = panel[1 + buf];
            }
            if (K == I) {
                // diagonal block pair: V = B_I B_I^T is symmetric — a SYRK: one job per 128-row block from its diagonal on, then
                // the lower triangle is mirrored (half the flops of the full block)
                const long long rows = (long long)ni * p.v;
                const int nrb = (int)((rows + 127) / 128);
                std::vector<XJob> jobs((size_t)nrb);
                long long t = 0;
                for (int r = 0; r < nrb; ++r) {
                    const long long r0 = (long long)r * 128, M = std::min<long long>(128, rows - r0), N = rows - r0;
                    GemmOut ov{};
                    ov.base = V + r0 * p.ldv + r0, ov.ld_m = p.ldv, ov.M = (int)M, ov.inner = (int)p.ldv, ov.valid_inner = (int)N, ov.stride_outer = 0;
                    ov.n_lin_total = N;
                    const double* Br = panel[0] + r0 * p.naux_ld;
                    CAN_TRY(gemm_job(jobs[r], Br, M, Br, N, p.naux, p.naux_ld, ov));
                    jobs[r].tile_begin = (int)t;
                    t += (long long)jobs[r].m_tiles * jobs[r].n_tiles;
                }
                CAN_CUDA(cudaMemcpyAsync(arena, jobs.data(), jobs.size() * sizeof(XJob), cudaMemcpyHostToDevice, st));
                CAN_TRY(launch_xform_gemm(false, reinterpret_cast<const XJob*>(arena), nrb, (int)t, p.num_sms, st));
                CAN_TRY(launch_mirror_lower(V, rows, p.ldv, st));
            } else {
                XJob J;
                GemmOut ov{};
                ov.base = V, ov.ld_m = p.ldv, ov.M = ni * p.v, ov.inner = (int)p.ldv, ov.valid_inner = nk * p.v, ov.stride_outer = 0;
                ov.n_lin_total = (long long)nk * p.v;
                CAN_TRY(gemm_job(J, panel[0], (long long)ni * p.v, PK, (long long)nk * p.v, p.naux, p.naux_ld, ov));
                CAN_CUDA(cudaMemcpyAsync(arena, &J, sizeof J, cudaMemcpyHostToDevice, st));
                CAN_TRY(launch_xform_gemm(false, reinterpret_cast<const XJob*>(arena), 1, J.m_tiles * J.n_tiles, p.num_sms, st));
            }
            if (buf >= 0) CAN_CUDA(cudaEventRecord(p.ev_free[buf], st));
            canonical_energy_kernel<<<CAN_GRID, 256, 0, st>>>(V, ni, nk, p.v, p.ldv, e_occ + i0, e_occ + k0, e_vir, K == I ? 1.0 : 2.0, slots);
            note_launch();
            CAN_CUDA(cudaGetLastError());
        }
    }
    ReduceCluster rc{};
    rc.gpart = slots;
    rc.E_out = E_out;
    rc.o = 1, rc.o8 = 1, rc.nslots = CAN_GRID;
    CAN_CUDA(cudaMemcpyAsync(ws + p.off_rc, &rc, sizeof rc, cudaMemcpyHostToDevice, st));
    return launch_reduce(reinterpret_cast<const ReduceCluster*>(ws + p.off_rc), 1, st);
}

int sie_dfmp2_canonical_info(sie_dfmp2_canon_t plan, long long* info, int n) {
    if (!plan) return 0;
    const long long vals[4] = {plan->Ib, plan->pblk, (plan->o + plan->Ib - 1) / plan->Ib, (long long)plan->panel_bytes};
    for (int i = 0; i < n && i < 4; ++i)
        if (info) info[i] = vals[i];
    return 4;
}

int sie_dfmp2_canonical_destroy(sie_dfmp2_canon_t plan) {
    if (!plan) return SIE_OK;
    if (plan->copy_stream) {
        cudaStreamSynchronize(plan->copy_stream);
        for (int i = 0; i < 2; ++i) {
            cudaEventDestroy(plan->ev_ready[i]);
            cudaEventDestroy(plan->ev_free[i]);
        }
        cudaEventDestroy(plan->ev_fork);
        cudaStreamDestroy(plan->copy_stream);
    }
    delete plan;
    return SIE_OK;
}

}  // extern "C"
