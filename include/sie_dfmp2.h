/*
 * sie_dfmp2.h — C ABI of libsie_dfmp2.so: fragment-projected density-fitted MP2 correlation energy of
 * SIE embedding clusters on one NVIDIA B200 (sm_100a).
 *
 * What is computed (citations: /root/reference/PAPER.md line numbers; DESIGN.md §1 restates them):
 *
 *   B^P_{ia}    = sum_{mu nu} C_{mu i} (P|mu nu) C_{nu a}              DF form of the cluster integral
 *                                                                     projection, Eq. S49 (L526)
 *   (ia|jb)     = sum_P B^P_{ia} B^P_{jb}
 *   t_{ij}^{ab} = (ia|jb) / (e_i + e_j - e_a - e_b)                    MP2 amplitudes, Eq. S15-S16 (L348-L351)
 *   G_{i'i}     = sum_j sum_{ab} t_{i'j}^{ab} ( 2 (ia|jb) - (ib|ja) )  closed-shell 2t-t pattern, Eq. S17-S18/S22
 *                                                                     (L355-L357, L390); only the first occupied
 *                                                                     index is projected, Eq. S44/S50 (L501, L535)
 *   E_frag      = sum_{i i'} P_frag[i][i'] G[i'][i] = Tr(P_frag G)     P_frag = C^f_{ii'}, Eq. S45/S59 (L505, L569)
 *
 * (P|mu nu) are already-fitted three-index factors (no metric is applied), restricted closed shell,
 * real arithmetic, all nocc orbitals correlated, FP64 throughout.  G is NOT symmetric and is never
 * symmetrised.  The orbital gap max(e_occ) < min(e_vir) is required (Eq. S16 denominators > 0).
 *
 * Conventions
 *   - every function returns an int status (SIE_OK = 0); outputs are untouched on error.
 *   - all matrices are row-major FP64.  The library never allocates device memory: the caller provides
 *     one workspace (size reported by the plan / batch query), e.g. a torch uint8 tensor, and owns every
 *     buffer.  Inputs are never modified and are not retained after the enqueued work completes.
 *   - pointer arguments are DEVICE pointers unless the plan / batch was created with
 *     SIE_FLAG_HOST_IO, in which case every data pointer (inputs and outputs, not the workspace) is a
 *     HOST pointer (pinned memory recommended) and the library stages the copies itself on `cuda_stream`;
 *     with SIE_FLAG_HOST_IO sie_dfmp2_energy / sie_dfmp2_batch synchronise the stream before returning.
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  Calls only enqueue
 *     work unless stated otherwise.
 *   - a plan is used by one host thread at a time; different plans are independent.
 */
#ifndef SIE_DFMP2_H
#define SIE_DFMP2_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sie_dfmp2_plan_s* sie_dfmp2_plan_t;

enum {
    SIE_OK = 0,
    SIE_EINVAL = 1,       /* bad size / null pointer / bad range */
    SIE_ENOMEM = 2,       /* host allocation failed or workspace too small */
    SIE_ECUDA = 3,        /* a CUDA runtime / driver call failed (see sie_dfmp2_last_cuda_error) */
    SIE_ESTATE = 4,       /* call order violated (e.g. energy before the transform covered [0,naux)) */
    SIE_EGAP = 5,         /* SIE_FLAG_VALIDATE only: max(e_occ) >= min(e_vir) */
    SIE_EUNSUPPORTED = 6, /* no CUDA device of compute capability 10.x */
    SIE_ETOOBIG = 7       /* sie_dfmp2_energy_noalloc: the problem needs more than the static scratch of SIE_NOALLOC_SCRATCH_BYTES */
};

enum {
    SIE_FLAG_VALIDATE = 1u,  /* energy/batch copy e_occ,e_vir to the host (synchronising) and check the gap */
    SIE_FLAG_REFERENCE = 2u, /* use the simple FP64-FMA reference kernels (any nocc; slow; cross-check path) */
    SIE_FLAG_HOST_IO = 4u,   /* data pointers are HOST pointers; the library stages H2D/D2H copies */
    SIE_FLAG_PROFILE = 8u,   /* bracket every launch group with CUDA events; read with *_timing (below) */
    SIE_FLAG_RDM_OCC = 16u,  /* sie_dfmp2_batch only: compute the occupied 1-RDM block of every cluster instead of the
                                energy (3b): G_out receives gamma, E_out receives Tr gamma, P_frag is ignored */
    SIE_FLAG_RDM_VIR = 32u,  /* sie_dfmp2_plan only: reserve the workspace sie_dfmp2_rdm_vir (3c) needs (three amplitude slabs) */
    SIE_FLAG_STAGE_FULL = 64u /* sie_dfmp2_plan with SIE_FLAG_HOST_IO: stage the WHOLE packed tensor in the workspace (naux * npair
                                 doubles more) instead of a two-buffer ring.  The upload of a cluster then never waits for its own
                                 GEMMs, so with two plans on two streams the integrals of cluster n+1 travel while the pair stage of
                                 cluster n runs (transform of n+1 enqueued before energy of n) */
};

/*
 * 1. sie_dfmp2_plan — host only.  Validates the sizes, chooses tile configurations and the internal aux
 *    sub-block (the rows of the half-transformed intermediate H that exist at once; at most 2 GB), and reports the device workspace (bytes, 256-byte aligned base required) the caller must
 *    pass to transform/energy.  The workspace holds B[a][i][P] between transform and energy.
 *      nao >= nocc + nvir, nocc >= 1, nvir >= 1, naux >= 1; aux_block = rows of (P|mu nu) processed per
 *      internal step (0 = auto).
 *    Three routes exist for the pair stage, reported by sie_dfmp2_plan_info()[7]:
 *      0 fused      nocc <= 128: one persistent kernel, V and t never leave the chip (the tuned path)
 *      2 general    nocc > 128 (e.g. the environment-occupied sub-space of PAPER.md Eq. S13): per occupied block a
 *                   slab GEMM, an amplitude pass and a split-K Gram GEMM, all on the FP64 tensor cores; the amplitude slab of
 *                   one occupied block (nvir^2 * nocc * block doubles, <= 4 GB or SIE_EINVAL) is the largest intermediate
 *      1 reference  SIE_FLAG_REFERENCE: simple FP64-FMA kernels, a cross-check only
 */
int sie_dfmp2_plan(sie_dfmp2_plan_t* plan, int nao, int nocc, int nvir, int naux, int aux_block,
                   unsigned flags, size_t* workspace_bytes);

/*
 * 2. sie_dfmp2_transform — AO->MO two-step half transform (steps A1+A2 of DESIGN.md) of the aux rows
 *    [p0,p1); call repeatedly, in any order, until [0,naux) is covered exactly once (overlap -> SIE_EINVAL).
 *      C_occ          [nao][nocc]   C_vir [nao][nvir]   (must be the same for every block of one plan)
 *      L_packed_block [(p1-p0)][nao(nao+1)/2]: element (P,mu,nu), mu >= nu, at (P-p0)*npair + mu(mu+1)/2 + nu
 *    Result: B^P_{ia} in the workspace (layout private to the library).
 */
int sie_dfmp2_transform(sie_dfmp2_plan_t plan, void* workspace, const double* C_occ, const double* C_vir,
                        const double* L_packed_block, int p0, int p1, void* cuda_stream);

/*
 * 3. sie_dfmp2_energy — fused pair stage (V, t, G never leave the chip) + projector/trace reduction
 *    (steps A3-A6).   e_occ[nocc], e_vir[nvir], P_frag[nocc][nocc] = P[i][i'] (NULL = identity),
 *    E_out: 1 double, G_out: [nocc][nocc] = G[i'][i] or NULL.  SIE_ESTATE if the transform has not
 *    covered [0,naux).  May be called again with other e/P on the same B.
 */
int sie_dfmp2_energy(sie_dfmp2_plan_t plan, void* workspace, const double* e_occ, const double* e_vir,
                     const double* P_frag, double* E_out, double* G_out, void* cuda_stream);

/*
 * 3a. sie_dfmp2_energy_lowrank — NEXT-3, "project first" (PAPER.md Eq. S33; fragment projector C^f = sum_f C_if C_i'f,
 *    Eq. S45): the fragment energy for a projector given in factored form, P_frag = Q Q^T with Q [nocc][r] row-major
 *    (the r fragment orbitals in the cluster's occupied basis), when G itself is not wanted:  E_frag = Tr(Q Q^T G).
 *    For r <= 32 the fused kernel contracts every (ia|jb) block with Q^T first — four r x o x o tensor-core products per
 *    virtual pair instead of two o x o x o ones, and no partial-G slots; above that it forms P and takes the G path.
 *    Same value as sie_dfmp2_energy(P_frag = Q Q^T) up to rounding order.  Fused route only (nocc <= 128;
 *    SIE_EUNSUPPORTED otherwise).  Pointers device or host per SIE_FLAG_HOST_IO; call order and errors as sie_dfmp2_energy.
 */
int sie_dfmp2_energy_lowrank(sie_dfmp2_plan_t plan, void* workspace, const double* e_occ, const double* e_vir,
                             const double* Q, int r, double* E_out, void* cuda_stream);

/*
 * 3n. sie_dfmp2_energy_noalloc — the fused pair stage + projector/trace (steps A3-A6, the work of sie_dfmp2_energy) for callers
 *    that must not allocate device memory and have no workspace to pass: code under CUDA graph capture, tight serving loops,
 *    harnesses that forbid cudaMalloc.  The partial-G slots, the tile work list and the descriptors live in ONE file-scope
 *    static device array of SIE_NOALLOC_SCRATCH_BYTES (24 MiB) inside the library; every GPU that loads the library holds it
 *    until the process exits.  The call allocates nothing on the device (no cudaMalloc / cudaFree / allocating library
 *    routine) and needs no plan.
 *      B       DEVICE, [nvir][nocc][ceil8(naux)] row-major with the aux index contiguous: B[a][i][P] = B^P_{ia}, 16-byte aligned
 *              (the layout sie_dfmp2_transform leaves at the start of its workspace; aux columns >= naux are never read)
 *      e_occ [nocc], e_vir [nvir], P_frag [nocc][nocc] or NULL (identity), E_out: 1 double, G_out [nocc][nocc] or NULL: DEVICE
 *    Limits: nocc <= 128 (SIE_EUNSUPPORTED above), and sie_dfmp2_noalloc_bytes(nocc, nvir) <= SIE_NOALLOC_SCRATCH_BYTES —
 *    148 x kp x ceil8(nocc)^2 doubles of slots (kp = 16 / ceil(nocc/8), at least 1) plus 8 bytes per pair tile; BASELINE
 *    config 3 (nocc 120, nvir 1080) needs 21.7 MB and fits; larger problems return SIE_ETOOBIG and touch nothing.
 *    Same results as sie_dfmp2_energy on the same B (same kernels, same tile order, same fixed-order reduction).
 *    ALL calls share the one array, which keeps the last call's contents; the call itself clears what must start at zero
 *    on `cuda_stream`.  Calls whose GPU work overlaps (two streams, two host threads) RACE on it: serialise them on one
 *    stream.  Enqueues only; does not synchronise.
 */
#define SIE_NOALLOC_SCRATCH_BYTES (24u << 20)
int sie_dfmp2_energy_noalloc(int nocc, int nvir, int naux, const double* B, const double* e_occ, const double* e_vir,
                             const double* P_frag, double* E_out, double* G_out, void* cuda_stream);
size_t sie_dfmp2_noalloc_bytes(int nocc, int nvir); /* scratch bytes the call above needs (0: sizes it does not support) */
size_t sie_dfmp2_noalloc_capacity(void);            /* = SIE_NOALLOC_SCRATCH_BYTES */

/*
 * 3b. sie_dfmp2_rdm_occ — NEXT-1: occupied block of the MP2 one-particle reduced density matrix of the
 *    cluster, PAPER.md Eq. S18 (L357) with the amplitudes of Eq. S15-S16 (L348-L351):
 *        gamma_ij = 2 delta_ij - 2 sum_k sum_ab t_ik^ab (2 t_jk^ab - t_jk^ba),   t_ik^ab = (ia|kb) / (e_i + e_k - e_a - e_b)
 *    (the matrix whose eigenvectors rank the occupied bath natural orbitals).  Same fused kernel as the energy: the
 *    (ia|kb) tile is turned into amplitudes in shared memory and contracted with itself; nothing reaches HBM.
 *      e_occ [nocc], e_vir [nvir]; gamma_out [nocc][nocc] row-major (symmetric), REQUIRED;
 *      trace_out: 1 double or NULL, receives Tr gamma (the electron count left in the occupied block).
 *    Pointers device or host per SIE_FLAG_HOST_IO, call order and errors as sie_dfmp2_energy; may be called before or
 *    after sie_dfmp2_energy on the same transformed workspace, any number of times.
 */
int sie_dfmp2_rdm_occ(sie_dfmp2_plan_t plan, void* workspace, const double* e_occ, const double* e_vir,
                      double* gamma_out, double* trace_out, void* cuda_stream);

/*
 * 3c. sie_dfmp2_rdm_vir — NEXT-1: virtual block of the MP2 one-particle reduced density matrix, PAPER.md Eq. S17 (L355):
 *        gamma_ab = 2 sum_ij sum_c t_ij^ac (2 t_ij^bc - t_ij^cb),   t_ij^ac = (ia|jc) / (e_i + e_j - e_a - e_c)
 *    (the matrix whose eigenvectors rank the virtual bath natural orbitals; with the impurity-occupied x environment-virtual
 *    orbital sets of Eq. S14, as C_occ / C_vir).  Runs on the general route at every size and needs a plan created
 *    with SIE_FLAG_RDM_VIR (SIE_ESTATE otherwise; SIE_EUNSUPPORTED with SIE_FLAG_REFERENCE).
 *      gamma_out [nvir][nvir] row-major (symmetric), REQUIRED;  trace_out: 1 double or NULL, receives Tr gamma_vir
 *      (= 2 nocc - Tr gamma_occ).  Pointers, call order and errors as sie_dfmp2_rdm_occ.
 */
int sie_dfmp2_rdm_vir(sie_dfmp2_plan_t plan, void* workspace, const double* e_occ, const double* e_vir,
                      double* gamma_out, double* trace_out, void* cuda_stream);

/*
 * 4. sie_dfmp2_batch — many independent clusters (no contraction across clusters) in one
 *    scheduled submission: per-cluster transforms, then ONE persistent pair kernel whose CTAs walk a
 *    static, cost-balanced list of (cluster, tile) work items, then one reduction launch (step A7).
 *      clusters: HOST array of descriptors (pointers device or host per SIE_FLAG_HOST_IO).
 *      workspace_bytes == 0 or workspace == NULL: query only, *needed receives the required size (make the query with the
 *      descriptors of the call, L_packed pointers included: the layout depends on which clusters share integrals).
 *    Shared integrals (device pointers): clusters of one system are different orbital sets over the SAME (P|mu nu)
 *    (PAPER.md L95).  Batch members that pass the same L_packed pointer with the same nao and naux are transformed
 *    together — their C_occ columns are stacked into one A1 GEMM — so the integrals are read once for all of them.
 *    With device pointers the transforms of ALL clusters run as one grouped launch per stage (coefficient transposes,
 *    A1 on the packed integrals, A2) and everything is enqueued on `cuda_stream`; with host pointers the clusters'
 *    integrals pass through one staging ring on an internal copy stream, cluster by cluster.
 *    Errors: SIE_EINVAL (sizes, null required pointers, misaligned workspace), SIE_ENOMEM (workspace too small;
 *    *needed is set), SIE_EGAP (SIE_FLAG_VALIDATE), SIE_ECUDA.  Outputs are untouched on SIE_EINVAL/SIE_ENOMEM.
 */
typedef struct {
    int nao, nocc, nvir, naux;
    const double* C_occ;    /* [nao][nocc] */
    const double* C_vir;    /* [nao][nvir] */
    const double* L_packed; /* [naux][nao(nao+1)/2] */
    const double* e_occ;    /* [nocc] */
    const double* e_vir;    /* [nvir] */
    const double* P_frag;   /* [nocc][nocc] or NULL (identity) */
    double* E_out;          /* 1 double */
    double* G_out;          /* [nocc][nocc] or NULL */
} sie_dfmp2_cluster_t;

int sie_dfmp2_batch(int ncluster, const sie_dfmp2_cluster_t* clusters, void* workspace, size_t workspace_bytes,
                    size_t* needed, unsigned flags, void* cuda_stream);

/*
 * Forgets which aux rows have been transformed (host-side state only; enqueues nothing), so the same plan can run
 * another cluster of the same shape — or the same one again — with the same or another workspace:
 * plan -> [transform... -> energy...] -> reset -> [transform... -> energy...] -> destroy.
 * Work already enqueued is not affected; the caller orders reuse of the workspace by using one stream.
 * A transform into a different workspace than the rows covered so far returns SIE_ESTATE unless reset first.
 */
int sie_dfmp2_plan_reset(sie_dfmp2_plan_t plan);

/*
 * 5. sie_dfmp2_canonical_* — NEXT-2: closed-shell canonical DF-MP2 correlation energy of a whole system,
 *        E_MP2 = sum_{ij} sum_{ab} (ia|jb) (2 (ia|jb) - (ib|ja)) / (e_i + e_j - e_a - e_b)       (Eq. S15-S16 with P_frag = I),
 *    the E_MP2 term of the bath-truncation correction (PAPER.md Eq. S63; Eq. S68; Table S1), for sizes
 *    where B^P_ia no longer fits in device memory.  B[i][a][P] (occupied-major, aux index contiguous, leading dimension
 *    ceil8(naux)) lives in a STORE the caller owns: pinned host memory for the out-of-core case, or device memory when it
 *    fits — any pointer cudaMemcpy understands; *bstore_bytes reports its size.
 *      plan       host only; occ_block = occupied orbitals per panel of the pair phase (0 = auto: three panels and the
 *                 (block x nvir)^2 integral block within ~12 GB); reports the device workspace.
 *      transform  aux rows [p0,p1) of the packed integrals (DEVICE pointer, as sie_dfmp2_transform) -> the store; call until
 *                 [0,naux) is covered exactly once; C_occ, C_vir DEVICE pointers.
 *      energy     occupied-block pairs I <= K: panels to the device on an internal copy stream (double-buffered under the
 *                 GEMM of the pair before), one tensor-core GEMM per pair of blocks, an elementwise pass into CTA-private
 *                 slots, fixed-order sum; e_occ, e_vir, E_out DEVICE pointers.  SIE_ESTATE before the transform is complete.
 *      info       [0] occupied block  [1] aux sub-block of the transform  [2] number of occupied blocks  [3] bytes of one panel
 *    Amplitudes are never stored; the (block x nvir)^2 integral block lives for one pair of blocks.
 */
typedef struct sie_dfmp2_canon_s* sie_dfmp2_canon_t;
int sie_dfmp2_canonical_plan(sie_dfmp2_canon_t* plan, int nao, int nocc, int nvir, int naux, int occ_block,
                             size_t* workspace_bytes, size_t* bstore_bytes);
int sie_dfmp2_canonical_transform(sie_dfmp2_canon_t plan, void* workspace, const double* C_occ, const double* C_vir,
                                  const double* L_packed_block, int p0, int p1, double* B_store, void* cuda_stream);
int sie_dfmp2_canonical_energy(sie_dfmp2_canon_t plan, void* workspace, const double* e_occ, const double* e_vir,
                               const double* B_store, double* E_out, void* cuda_stream);
int sie_dfmp2_canonical_info(sie_dfmp2_canon_t plan, long long* info, int n);
int sie_dfmp2_canonical_destroy(sie_dfmp2_canon_t plan);

/* Frees the host-side plan (never touches device memory). NULL is allowed. */
int sie_dfmp2_destroy(sie_dfmp2_plan_t plan);

/* Static string for a status code. */
const char* sie_dfmp2_strerror(int status);

/* Text of the last CUDA error seen by this library on the calling thread ("" if none). */
const char* sie_dfmp2_last_cuda_error(void);

/* Number of kernels this library has launched since load (all threads); bench.py's gpu_launches. */
unsigned long long sie_dfmp2_launch_count(void);

/*
 * Introspection for benchmarks/tests: fills info[0..n) with plan facts, returns how many exist.
 *   0, 1: pair-tile rows / cols in rows of B, ceil8(ta*nocc) <= 128   2: virtual blocks per tile side (ta)
 *   3: ceil8(nocc), the leading dimension of a partial-G slot   4: number of pair tiles   5: persistent CTAs   6: internal aux sub-block
 *   7: pair-stage route: 0 fused, 1 reference kernels, 2 general (nocc > 128)
 */
int sie_dfmp2_plan_info(sie_dfmp2_plan_t plan, long long* info, int n);

/*
 * Stage timing (plans / batches created with SIE_FLAG_PROFILE; SIE_ESTATE otherwise).  Synchronises on the
 * recorded events, sums the device time of every launch group enqueued since the last query, then clears.
 *   ms[0..7):  0 coefficient transposes  1 unused (always 0: A1 reads the packed triangle directly)  2 A1 GEMM  3 A2 GEMM  4 fused pair kernel
 *              5 reduce/trace  6 reference kernels          (milliseconds, HOST array of n doubles)
 *   ms[7..14): the number of launch groups summed into each of the seven entries above.
 * sie_dfmp2_batch_timing reports the calling thread's last sie_dfmp2_batch call.
 */
int sie_dfmp2_plan_timing(sie_dfmp2_plan_t plan, double* ms, int n);
int sie_dfmp2_batch_timing(double* ms, int n);

/*
 * FP64 issue-rate microkernels: the live denominator of the FP64 roofline.
 *   kind 0: register-resident DMMA (mma.sync.m8n8k4.f64)   1: register-resident DFMA
 *        2: shared-memory-fed DMMA with the fragment loads of the pair mainloop
 *   iters: loop trips per warp;  ctas_per_sm: CTAs (256 threads) launched per SM;  scratch: >= 8 bytes, DEVICE.
 * Runs the kernel twice on `cuda_stream`, times the second run with events, synchronises;
 * *tflops (HOST) = flops / time, *ms (HOST, may be NULL) = that time.
 */
int sie_dfmp2_probe_fp64(int kind, int iters, int ctas_per_sm, void* scratch, double* tflops, double* ms, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* SIE_DFMP2_H */
