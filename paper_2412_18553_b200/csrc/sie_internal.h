// sie_internal.h — host-side launcher declarations shared by the translation units of libsie_dfmp2.so.
#pragma once

#include <cuda.h>
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

namespace sie {

// ---- transform.cu ------------------------------------------------------------------------------
struct GemmOut {
    double* base;          // output base pointer
    long long ld_m;        // offset per row m
    int M;                 // valid rows
    int inner;             // n_lin -> (outer = n_lin / inner, rem = n_lin % inner)
    int valid_inner;       // column valid iff rem < valid_inner
    long long stride_outer;  // offset = outer * stride_outer + rem
    long long n_lin_total;   // column valid iff n_lin < n_lin_total
    int accumulate;          // 1: C += (read-modify-write; every element has one owner per launch), 0: C =
};
// One GEMM of a grouped launch: C[m][n] = sum_k A[m][k] * Bop[n][k], K-major operands (transform.cu)
struct alignas(128) XJob {
    CUtensorMap mapA;       // K-major A operand [M][K], box {8, 8*m8, 1}
    CUtensorMap mapB;       // TMA mode: K-major Bop [N][K], box {8, 128, 1}
    const double* Lp;       // packed mode: [np][npair]
    long long npair;
    long long n_total;      // valid flat columns n
    int nao;                // packed mode: n = P * nao + nu
    int M, m8, m_tiles, n_tiles, kblocks;
    int k0_blocks;          // first K-block of this job (split-K jobs share their tensor maps)
    int b_c1_off, b_c1_mul, b_c2_mul;  // TMA mode: N-tile nb of Bop sits at coordinates (k, b_c1_off + nb * b_c1_mul, nb * b_c2_mul)
    int tile_begin;         // global index of this job's first tile (tiles of a job: m fastest)
    GemmOut out;
};

int launch_xform_gemm(bool packed, const XJob* d_jobs, int njobs, int total_tiles, int num_sms, cudaStream_t st);
// one coefficient transpose of a grouped launch: out[c][r] = in[r][c] for r < rows, c < cols, leading dimension ld_out
struct TJob {
    const double* in;
    double* out;
    int rows, cols, ld_out, pad;
};
int launch_transpose_jobs(const TJob* d_jobs, int njobs, int max_rows, int max_cols, cudaStream_t st);

// descriptor / small-operand writers that do not use the host-to-device copy engine (see transform.cu)
int launch_poke(const void* payload, size_t nbytes, void* dst, cudaStream_t st);      // nbytes <= 512, multiple of 8
int launch_copy_f64(const double* src, double* dst, size_t n, cudaStream_t st);       // src device or mapped pinned host

// ---- pair.cu -----------------------------------------------------------------------------------
struct alignas(128) PairCluster {  // one per cluster, lives in the workspace (global memory)
    CUtensorMap map;               // B as the plain matrix {naux, nocc*nvir, 1}, box {8, t8, 1}
    const double* e_occ;
    const double* e_vir;
    double* gpart;                 // partial-G slots of this cluster: [ncta][kp][o8*o8]
    int o, v, o8, ta;              // o8 = ceil8(o): leading dimension of a partial-G slot; ta virtual blocks per tile edge
    int kblocks;                   // ceil(naux / 8)
    int kp;                        // epilogue sub-block split parts
    uint32_t tx_bytes;             // bytes of both operand boxes of one stage
    int t8;                        // tile edge in rows of B: ceil8(ta * o) <= 128
    int gate;                      // 1: producers keep the CTAs of a round in K-lockstep (equal-cost tiles only)
    int mode;                      // 0: G of the energy path; 1: Gamma of the occupied 1-RDM block (amplitudes on both sides)
    const double* Qt;              // mode 2 (energy only, P_frag = Q Q^T of rank r <= 32): Q^T, zero padded, [8*r8][ldq]
    int r8, ldq;                   //   gpart then holds per-warp partial energies [ncta][16] instead of G slots
};
struct PairTile {                  // 8 bytes
    int cluster;
    unsigned short bi, bj;         // virtual-block indices, bi <= bj
};
struct PairGeom {                  // tile configuration facts for host-side planning
    int TM, TN, ncons;
};
PairGeom pair_geom();
// Energy-mode launches that contain a cluster with nocc <= this use the kernel instantiation whose strips of such clusters
// are epilogue_strip_small (launch_pair mode 3).  Measured (custom:o,4o,1536): small strips +4...5.5 % at o = 72...96,
// -1 % at 104, -5 % at 112, -6 % at 120, equal at 128 — so larger blocks keep the generic strip in either instantiation.
constexpr int PAIR_SMALL_STRIP_MAX_O = 96;
// In the polling-producer kernels (pair_producer_warp() != 0) the small strips also win above 96: the loss at o = 104...120 came
// from the strips' timing delaying warp 0, the producer AND pace-setter of the old placement; with the producer on warp 12
// config 3 (o = 120) goes 0.928 -> 0.940 with them, o = 104 +1.5 %, o = 112 +-0.
constexpr int PAIR_SMALL_STRIP_MAX_O_POLL = 120;
inline bool pair_small_strip(int o, bool poll) { return o <= (poll ? PAIR_SMALL_STRIP_MAX_O_POLL : PAIR_SMALL_STRIP_MAX_O); }
size_t pair_smem_bytes();
// mode: 0 energy path (G), 1 occupied 1-RDM block (Gamma), 2 energy only with a low-rank projector, 3 = mode 0 through the
// instantiation whose strips for o <= 64 are epilogue_strip_small (same sums; chosen by the caller when such clusters exist); one mode per launch
// producer_warp: the math warp whose lane 0 issues the TMA loads (pair_producer_warp() for a tile edge t8)
int launch_pair(const PairCluster* d_clusters, const PairTile* d_tiles, int ntiles, int ncta, int tmax, int mode, int producer_warp,
                cudaStream_t st);
// Tile edges that are not a multiple of 32 rows give the 4 x 4 warp grid uneven rectangles: warp 12 = (3,3) then owns the
// smallest one and runs ahead of the others, which is where the producer lane belongs (it refills while it waits for its
// own data); with even rectangles every warp has the same work and the producer stays on warp 0, topping up once per step.
inline int pair_producer_warp(int t8) { return ((t8 >> 3) & 3) ? 12 : 0; }

struct ReduceCluster {             // per cluster, device array
    const double* gpart;           // [nslots][o8*o8]
    const double* P;               // [o][o] or nullptr
    double* E_out;                 // 1
    double* G_out;                 // [o][o] or nullptr
    int o, o8, nslots;
    int mode;                      // 0: G_out = G, E_out = sum P o G^T; 1: G_out = 2 delta - 2 Gamma, E_out = its trace;
                                   // 2: G_out = 2 * sum (virtual block gamma_ab, Eq. S17), E_out = its trace
};
int launch_reduce(const ReduceCluster* d_rc, int ncluster, cudaStream_t st);
// Q [o][r] -> Qt (Q^T zero padded to [8*r8][ldq]) when Qt != nullptr, and P = Q Q^T [o][o] when P != nullptr
int launch_lowrank_prep(const double* Q, int o, int r, double* Qt, int ldq, int r8, double* P, cudaStream_t st);

// ---- general.cu --------------------------------------------------------------------------------
// Any-size pair stage (nocc > 128, and gamma_vir at every size): slab GEMM -> combine -> split-K Gram GEMM per occupied block.
struct GeneralGeom {
    int Kb, ldc;                 // occupied block (power of two), leading dimension of a slab row = ceil8(v * Kb)
    int nsplit_occ, nsplit_vir;  // K splits (= partial slots) of the Gram GEMM of the occupied / virtual block
    int max_jobs;                // job descriptors per occupied block
    bool ok;                     // false: one slab would exceed 4 GB (sizes beyond this route)
    bool full;                   // one occupied block covers the cluster: the slab GEMM is a SYRK (upper tiles + mirror)
    size_t slab_bytes, slots_bytes;
};
GeneralGeom general_geom(int o, int v, int num_sms);
size_t general_scratch_bytes(const GeneralGeom& g, int o);
// mode 0: G (energy path), 1: Gamma_occ, 2: gamma_vir / 2.  Partial results in slots [*nslots][n*n], n = o (modes 0, 1) or v.
int general_pair(const GeneralGeom& g, const double* Bmat, int o, int v, int naux, int naux_ld, const double* e_occ, const double* e_vir,
                 int mode, unsigned char* scratch, double* slots, int* nslots, int num_sms, cudaStream_t st);

// V[r][c] = V[c][r] for r > c of a square n x n matrix (leading dimension ld) whose upper triangle was computed
int launch_mirror_lower(double* V, long long n, long long ld, cudaStream_t st);

// ---- ref_kernels.cu ----------------------------------------------------------------------------
// Simple FP64-FMA kernels following the definition step by step (any nocc). B layout [v][o][naux_ld].
int ref_transform(const double* C_occ, const double* C_vir, const double* Lp_block, int nao, int o, int v, int p0, int p1,
                  double* H /*[(p1-p0)][o][nao]*/, double* B, int naux_ld, cudaStream_t st);
int ref_pair(const double* B, int o, int v, int naux, int naux_ld, const double* e_occ, const double* e_vir,
             double* Vj /*[o][v][v]*/, double* G /*[o][o]*/, int mode /*0 G, 1 Gamma*/, cudaStream_t st);
size_t ref_vj_bytes(int o, int v);

// ---- probes.cu ---------------------------------------------------------------------------------
int run_probe(int kind, int iters, int ctas_per_sm, int num_sms, double* sink, double* flops, float* ms, cudaStream_t st);

}  // namespace sie
