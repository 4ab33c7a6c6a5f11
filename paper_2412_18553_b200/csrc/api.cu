// api.cu — the C-ABI boundary of libsie_dfmp2.so (include/sie_dfmp2.h): planning, workspace layout,
// tensor-map encoding, the static (cluster, tile) schedule, and the launch sequences.
#include <algorithm>
#include <atomic>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/sie_dfmp2.h"
#include "sie_common.cuh"
#include "sie_internal.h"

namespace sie {

// ------------------------------------------------------------------------------------------------ bookkeeping
static std::atomic<unsigned long long> g_launches{0};
static thread_local std::string g_last_error;

void note_launch() { g_launches.fetch_add(1, std::memory_order_relaxed); }
int set_cuda_error_text(const char* s) {
    g_last_error = s ? s : "";
    return SIE_ECUDA;
}
int set_cuda_error(cudaError_t e) {
    g_last_error = std::string(cudaGetErrorName(e)) + ": " + cudaGetErrorString(e);
    return SIE_ECUDA;
}
#define SIE_CUDA(call)                                   \
    do {                                                 \
        cudaError_t e__ = (call);                        \
        if (e__ != cudaSuccess) return set_cuda_error(e__); \
    } while (0)
#define SIE_TRY(call)                  \
    do {                               \
        int rc__ = (call);             \
        if (rc__ != SIE_OK) return rc__; \
    } while (0)

// ------------------------------------------------------------------------------------------------ tensor maps
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn get_encode_fn() {
    // function-local static: initialised once, thread-safe (C++11); the entry point is process-wide, not per device
    static const EncodeTiledFn fn = []() -> EncodeTiledFn {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            return reinterpret_cast<EncodeTiledFn>(p);
        return nullptr;
    }();
    return fn;
}

int ensure_smem_attr(const void* kernel, int bytes, SmemAttrOnce& once) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return set_cuda_error(e);
    const bool tracked = dev >= 0 && dev < 64;
    if (tracked && (__atomic_load_n(&once.done, __ATOMIC_ACQUIRE) >> dev & 1ull)) return SIE_OK;
    e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e != cudaSuccess) return set_cuda_error(e);
    if (tracked) __atomic_fetch_or(&once.done, 1ull << dev, __ATOMIC_RELEASE);
    return SIE_OK;
}

int make_tensor_map_3d(CUtensorMap* out, const double* base, uint64_t d0, uint64_t d1, uint64_t d2, uint64_t stride1_bytes,
                       uint64_t stride2_bytes, uint32_t b0, uint32_t b1, uint32_t b2) {
    EncodeTiledFn fn = get_encode_fn();
    if (!fn) return set_cuda_error_text("cuTensorMapEncodeTiled entry point not available");
    cuuint64_t dims[3] = {d0, d1, d2};
    cuuint64_t strides[2] = {stride1_bytes, stride2_bytes};
    cuuint32_t box[3] = {b0, b1, b2};
    cuuint32_t estr[3] = {1, 1, 1};
    CUresult r = fn(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, const_cast<double*>(base), dims, strides, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        char buf[256];
        snprintf(buf, sizeof buf,
                 "cuTensorMapEncodeTiled failed (%d): dims {%llu,%llu,%llu} strides {%llu,%llu} box {%u,%u,%u} base %p", (int)r,
                 (unsigned long long)d0, (unsigned long long)d1, (unsigned long long)d2, (unsigned long long)stride1_bytes,
                 (unsigned long long)stride2_bytes, b0, b1, b2, (const void*)base);
        return set_cuda_error_text(buf);
    }
    return SIE_OK;
}

// Facts of the CURRENT device (cudaGetDevice of the calling thread), cached per device ordinal in atomics:
// a process may drive several GPUs and several host threads may plan concurrently.
static std::atomic<int> g_dev_sms[64];    // 0 = not queried yet
static std::atomic<int> g_dev_major[64];  // 0 = not queried yet

static int query_num_sms() {
    int dev = 0, n = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) {
        (void)cudaGetLastError();
        return 148;  // planning without a device (CPU-only host): B200 value
    }
    const bool tracked = dev >= 0 && dev < 64;
    if (tracked && (n = g_dev_sms[dev].load(std::memory_order_relaxed)) > 0) return n;
    if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) {
        (void)cudaGetLastError();
        return 148;
    }
    if (tracked) g_dev_sms[dev].store(n, std::memory_order_relaxed);
    return n;
}

static int check_device() {
    int dev = 0, major = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return set_cuda_error(e);
    const bool tracked = dev >= 0 && dev < 64;
    if (!tracked || (major = g_dev_major[dev].load(std::memory_order_relaxed)) == 0) {
        e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
        if (e != cudaSuccess) return set_cuda_error(e);
        if (tracked) g_dev_major[dev].store(major, std::memory_order_relaxed);
    }
    return major == 10 ? SIE_OK : SIE_EUNSUPPORTED;
}

}  // namespace sie

using namespace sie;

// ------------------------------------------------------------------------------------------------ stage timing
// SIE_FLAG_PROFILE: every launch group is bracketed by a pair of events on the caller's stream; the
// elapsed times are summed per stage when queried (sie_dfmp2_plan_timing / sie_dfmp2_batch_timing).
enum { ST_COEFF = 0, ST_UNPACK, ST_T1, ST_T2, ST_PAIR, ST_REDUCE, ST_REF, ST_COUNT };
struct Prof {
    bool on = false;
    std::vector<cudaEvent_t> pool;
    struct Span { int stage, e0, e1; };
    std::vector<Span> spans;
    size_t used = 0;
    int take() {
        if (used == pool.size()) {
            cudaEvent_t e;
            if (cudaEventCreate(&e) != cudaSuccess) return -1;
            pool.push_back(e);
        }
        return (int)used++;
    }
    int begin(int stage, cudaStream_t st) {
        if (!on) return -1;
        const int a = take(), b = take();
        if (a < 0 || b < 0) return -1;
        cudaEventRecord(pool[a], st);
        spans.push_back(Span{stage, a, b});
        return (int)spans.size() - 1;
    }
    void end(int span, cudaStream_t st) {
        if (span >= 0) cudaEventRecord(pool[spans[span].e1], st);
    }
    void reset() {
        spans.clear();
        used = 0;
    }
    // sums per stage (ms) and launch-group counts; synchronises on the recorded events; then resets
    int collect(double* ms, double* counts) {
        for (int k = 0; k < ST_COUNT; ++k) ms[k] = counts[k] = 0.0;
        for (const Span& s : spans) {
            cudaError_t e = cudaEventSynchronize(pool[s.e1]);
            float t = 0.f;
            if (e == cudaSuccess) e = cudaEventElapsedTime(&t, pool[s.e0], pool[s.e1]);
            if (e != cudaSuccess) {
                reset();
                return set_cuda_error(e);
            }
            ms[s.stage] += t;
            counts[s.stage] += 1.0;
        }
        reset();
        return SIE_OK;
    }
    ~Prof() {
        for (cudaEvent_t e : pool) cudaEventDestroy(e);
    }
};
struct ProfSpan {  // RAII bracket
    Prof& p;
    cudaStream_t st;
    int id;
    ProfSpan(Prof& p_, int stage, cudaStream_t st_) : p(p_), st(st_), id(p_.begin(stage, st_)) {}
    ~ProfSpan() { p.end(id, st); }
};
static thread_local Prof g_batch_prof;

// ------------------------------------------------------------------------------------------------ plan
struct sie_dfmp2_plan_s {
    Prof prof;
    int nao = 0, o = 0, v = 0, naux = 0;
    unsigned flags = 0;
    bool ref = false, general = false, fused = true, has_gen = false;
    GeneralGeom gen{};
    size_t off_gen = 0, off_gslots = 0, off_Qt = 0;
    int nao_ld = 0, naux_ld = 0, o8 = 0, ta = 1, t8 = 8, nblk = 0, pblk = 0, cblk = 0, max_jobs = 0, ncta = 0, kp = 1, num_sms = 148;
    size_t npair = 0;
    std::vector<PairTile> tiles;  // cluster field = 0; rewritten when used inside a batch
    double tile_cost = 0;         // relative cost of one tile (for batch ordering)
    // workspace offsets (bytes)
    size_t off_B = 0, off_CoT = 0, off_CvT = 0, off_jobs = 0, off_H = 0, off_gpart = 0, off_desc = 0, off_tiles = 0, off_rc = 0,
           off_stage = 0, off_io = 0, off_refH = 0, off_refVj = 0, off_refG = 0, total = 0;
    size_t gpart_bytes = 0, stage_buf_bytes = 0;
    // io sub-offsets (doubles, relative to off_io)
    size_t io_Cocc = 0, io_Cvir = 0, io_eo = 0, io_ev = 0, io_P = 0, io_E = 0, io_G = 0, io_doubles = 0;
    // state
    std::vector<std::pair<int, int>> covered;
    long long covered_rows = 0;
    const void* c_ready_ws = nullptr;  // workspace for which the transposed coefficient copies are valid
    const void* tiles_ws = nullptr;    // workspace that holds the (static) tile list
    const double* dC_occ = nullptr;    // device pointers of the coefficients used by the transform
    const double* dC_vir = nullptr;
    // HOST_IO copy pipeline
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t ev_ready[2] = {nullptr, nullptr}, ev_consumed[2] = {nullptr, nullptr}, ev_fork = nullptr;
    int stage_turn = 0;
    bool stage_full = false;
    std::vector<cudaEvent_t> ev_chunk;  // SIE_FLAG_STAGE_FULL: one "chunk landed" event per staged chunk of a call
};

namespace {

struct Carver {
    size_t off = 0;
    size_t take(size_t bytes) {
        size_t r = off;
        off = align_up(off + bytes, 256);
        return r;
    }
};

void build_tiles(int nblk, std::vector<PairTile>& out) {
    // upper triangle bi <= bj, enumerated in column groups of S blocks so that the ~148 tiles in flight
    // share a dozen A panels and a dozen B panels (L2 reuse of the streamed operands)
    const int S = 12;
    out.clear();
    out.reserve((size_t)nblk * (nblk + 1) / 2);
    for (int J0 = 0; J0 < nblk; J0 += S) {
        const int J1 = std::min(nblk, J0 + S);
        for (int bi = 0; bi < J1; ++bi)
            for (int bj = std::max(bi, J0); bj < J1; ++bj) out.push_back(PairTile{0, (unsigned short)bi, (unsigned short)bj});
    }
}

enum { CARVE_NONE = 0, CARVE_MEMBER = 1, CARVE_ALL = 2 };  // what plan_init lays out beside B and the partial-G slots

int plan_init(sie_dfmp2_plan_s& p, int nao, int nocc, int nvir, int naux, int aux_block, unsigned flags, int carve) {
    if (nao < 1 || nocc < 1 || nvir < 1 || naux < 1 || aux_block < 0) return SIE_EINVAL;
    if ((long long)nocc + nvir > nao) return SIE_EINVAL;
    if (flags & ~(SIE_FLAG_VALIDATE | SIE_FLAG_REFERENCE | SIE_FLAG_HOST_IO | SIE_FLAG_PROFILE | SIE_FLAG_RDM_VIR | SIE_FLAG_STAGE_FULL))
        return SIE_EINVAL;
    if ((flags & SIE_FLAG_STAGE_FULL) && !(flags & SIE_FLAG_HOST_IO)) return SIE_EINVAL;
    p.nao = nao;
    p.o = nocc;
    p.v = nvir;
    p.naux = naux;
    p.flags = flags;
    p.npair = (size_t)nao * (nao + 1) / 2;
    p.num_sms = query_num_sms();
    const PairGeom geo = pair_geom();
    p.ref = (flags & SIE_FLAG_REFERENCE) != 0;
    p.general = !p.ref && nocc > geo.TM;  // an o x o block no longer fits one CTA tile: slab/Gram route (general.cu)
    p.fused = !p.ref && !p.general;
    p.nao_ld = (int)align_up((size_t)nao, 8);
    p.naux_ld = (int)align_up((size_t)naux, 8);
    p.o8 = (int)align_up((size_t)nocc, 8);
    // internal aux sub-block = the rows of H[i][P][nu] that exist at once between A1 and A2
    if (p.ref) {
        p.pblk = std::min(naux, aux_block > 0 ? aux_block : 64);
        p.cblk = p.pblk;
    } else {
        // at most 2 GB of H, and flat column indices (P, nu) and (i, P) of the two GEMMs below 2^31; each sub-block is ONE
        // grouped launch per stage, so there is no reason to make it smaller than that
        const size_t per_p = (size_t)nocc * p.nao_ld * 8;
        long long pb = std::max<long long>(8, (long long)(((size_t)2 << 30) / per_p));
        pb = std::min<long long>(pb, (long long)0x7fffffff / std::max(nao, nocc) - 1);
        if (aux_block > 0) pb = std::min<long long>(pb, aux_block);
        if (pb < naux) pb = std::max<long long>(8, pb / 8 * 8);
        p.pblk = (int)std::min<long long>(pb, naux);
        // HOST_IO: rows of packed (P|mu nu) per staging buffer (512 MB each, two of them)
        long long cb = std::max<long long>(8, (long long)(((size_t)512 << 20) / (p.npair * 8)) / 8 * 8);
        p.cblk = (int)std::min<long long>(cb, p.pblk);
    }
    if (p.fused) {
        // pair tiling: ta whole virtual blocks (ta*o <= 128 rows of B, o itself is never padded) per tile edge
        p.ta = std::max(1, geo.TM / nocc);
        p.t8 = (int)align_up((size_t)p.ta * nocc, 8);
        p.nblk = (nvir + p.ta - 1) / p.ta;
        if (p.nblk > 65535) return SIE_EINVAL;
        build_tiles(p.nblk, p.tiles);
        p.ncta = (int)std::min<size_t>((size_t)p.num_sms, p.tiles.size());
        const int nst = p.o8 / 8;
        p.kp = nst >= geo.ncons ? 1 : geo.ncons / nst;
        p.gpart_bytes = (size_t)p.num_sms * p.kp * p.o8 * p.o8 * 8;  // sized for any CTA count up to num_sms
        p.tile_cost = (double)p.t8 * p.t8 * naux + 4.0 * p.ta * p.ta * (double)p.o8 * p.o8 * p.o8;
    }
    // workspace
    Carver c;
    p.off_B = c.take((size_t)nvir * nocc * p.naux_ld * 8);
    if (p.fused)
        p.off_gpart = c.take(p.gpart_bytes);
    else if (p.ref)
        p.off_refG = c.take((size_t)nocc * nocc * 8);
    if (!p.ref && (p.general || (flags & SIE_FLAG_RDM_VIR))) {
        p.gen = general_geom(nocc, nvir, p.num_sms);
        if (!p.gen.ok) return SIE_EINVAL;  // one amplitude slab (nvir^2 * nocc doubles) would exceed 4 GB
        p.has_gen = true;
        p.off_gslots = c.take(p.gen.slots_bytes);
        if (carve == CARVE_ALL) p.off_gen = c.take(general_scratch_bytes(p.gen, nocc));
    }
    // job descriptors of one transform call: one A1 job per staged chunk (HOST_IO) or per sub-block, one A2 job per sub-block
    p.max_jobs = (naux + p.pblk - 1) / p.pblk + (naux + p.cblk - 1) / p.cblk + 8;
    if (carve == CARVE_MEMBER && !p.ref) {  // member of a device-pointer batch: private coefficient copies and H
        p.off_CoT = c.take((size_t)nocc * p.nao_ld * 8);
        p.off_CvT = c.take((size_t)nvir * p.nao_ld * 8);
        p.off_H = c.take((size_t)nocc * p.pblk * p.nao_ld * 8);
    }
    if (carve == CARVE_ALL) {
        if (!p.ref) {
            p.off_CoT = c.take((size_t)nocc * p.nao_ld * 8);
            p.off_CvT = c.take((size_t)nvir * p.nao_ld * 8);
            p.off_H = c.take((size_t)nocc * p.pblk * p.nao_ld * 8);
            p.off_jobs = c.take((size_t)p.max_jobs * sizeof(XJob) + 2 * sizeof(TJob));
            p.off_desc = c.take(sizeof(PairCluster));
            p.off_Qt = c.take((size_t)32 * p.o8 * 8 + (size_t)nocc * nocc * 8);  // Q^T of a low-rank projector, and P = Q Q^T
            p.off_tiles = c.take(p.tiles.size() * sizeof(PairTile) + 256);  // + the round-gate counter behind the list
        } else {
            p.off_refH = c.take((size_t)p.pblk * nocc * nao * 8);
            p.off_refVj = c.take(ref_vj_bytes(nocc, nvir));
        }
        p.off_rc = c.take(sizeof(ReduceCluster));
        if (flags & SIE_FLAG_HOST_IO) {
            p.stage_buf_bytes = align_up((size_t)p.cblk * p.npair * 8, 256);
            p.stage_full = (flags & SIE_FLAG_STAGE_FULL) && !p.ref;
            // two-buffer ring, or (SIE_FLAG_STAGE_FULL) room for the whole packed tensor so that the upload of a cluster never
            // waits for the GEMMs of an earlier chunk and can run under the pair stage of ANOTHER plan on another stream
            p.off_stage = c.take(p.stage_full ? align_up((size_t)naux * p.npair * 8, 256) : 2 * p.stage_buf_bytes);
            size_t d = 0;
            p.io_Cocc = d, d += (size_t)nao * nocc;
            p.io_Cvir = d, d += (size_t)nao * nvir;
            p.io_eo = d, d += nocc;
            p.io_ev = d, d += nvir;
            p.io_P = d, d += (size_t)nocc * nocc;
            p.io_E = d, d += 2;
            p.io_G = d, d += std::max((size_t)nocc * nocc, (flags & SIE_FLAG_RDM_VIR) ? (size_t)nvir * nvir : (size_t)0);
            p.io_doubles = d;
            p.off_io = c.take(d * 8);
        }
    }
    p.total = c.off;
    return SIE_OK;
}

int ensure_copy_pipeline(sie_dfmp2_plan_s& p) {
    if (p.copy_stream) return SIE_OK;
    SIE_CUDA(cudaStreamCreateWithFlags(&p.copy_stream, cudaStreamNonBlocking));
    for (int i = 0; i < 2; ++i) {
        SIE_CUDA(cudaEventCreateWithFlags(&p.ev_ready[i], cudaEventDisableTiming));
        SIE_CUDA(cudaEventCreateWithFlags(&p.ev_consumed[i], cudaEventDisableTiming));
    }
    SIE_CUDA(cudaEventCreateWithFlags(&p.ev_fork, cudaEventDisableTiming));
    return SIE_OK;
}

struct Scratch {  // transform scratch of one cluster (device pointers)
    double *CoT, *CvT, *H, *refH;
    unsigned char* jobs;   // arena of max_jobs XJob + 2 TJob descriptors
    unsigned char* stage;  // HOST_IO: 2 staging buffers
    size_t stage_buf_bytes;
};

// ---- job descriptors of the grouped transform GEMMs (transform.cu)
// A1 on `np` packed rows starting at Lq: H[i][P][nu] for P in [h0, h0+np) of an H sub-block that holds pbH rows
int make_a1_job(XJob& J, const sie_dfmp2_plan_s& p, const double* CoT, const double* Lq, int np, double* H, int h0, int pbH) {
    std::memset(&J, 0, sizeof J);
    const int m_tiles = (p.o + 127) / 128;
    const int m8 = ((p.o + m_tiles - 1) / m_tiles + 7) / 8;  // o is cut into m_tiles near-equal chunks of 8*m8 <= 128 rows
    SIE_TRY(make_tensor_map_3d(&J.mapA, CoT, p.nao, p.o, 1, (uint64_t)p.nao_ld * 8, (uint64_t)p.nao_ld * 8 * p.o, 8, 8 * m8, 1));
    J.Lp = Lq;
    J.npair = (long long)p.npair;
    J.nao = p.nao;
    J.n_total = (long long)np * p.nao;
    J.M = p.o;
    J.m8 = m8;
    J.m_tiles = (p.o + 8 * m8 - 1) / (8 * m8);
    J.n_tiles = (int)((J.n_total + 127) / 128);
    J.kblocks = (p.nao + 7) / 8;
    J.out.base = H + (size_t)h0 * p.nao_ld;
    J.out.ld_m = (long long)pbH * p.nao_ld;
    J.out.M = p.o;
    J.out.inner = p.nao;
    J.out.valid_inner = p.nao;
    J.out.stride_outer = p.nao_ld;
    J.out.n_lin_total = J.n_total;
    return SIE_OK;
}
// A2 on an H sub-block of pb aux rows starting at aux index q0: B[a][i][q0+P] = sum_nu CvT[a][nu] * H[(i,P)][nu]
int make_a2_job(XJob& J, const sie_dfmp2_plan_s& p, const double* CvT, const double* H, int pb, double* Bmat, int q0) {
    std::memset(&J, 0, sizeof J);
    const int m_tiles = (p.v + 127) / 128;
    const int m8 = ((p.v + m_tiles - 1) / m_tiles + 7) / 8;  // v is cut into m_tiles near-equal chunks of 8*m8 <= 128 rows
    SIE_TRY(make_tensor_map_3d(&J.mapA, CvT, p.nao, p.v, 1, (uint64_t)p.nao_ld * 8, (uint64_t)p.nao_ld * 8 * p.v, 8, 8 * m8, 1));
    SIE_TRY(make_tensor_map_3d(&J.mapB, H, p.nao, (uint64_t)p.o * pb, 1, (uint64_t)p.nao_ld * 8, (uint64_t)p.nao_ld * 8 * p.o * pb, 8,
                               128, 1));
    J.n_total = (long long)p.o * pb;
    J.b_c1_mul = 128;
    J.M = p.v;
    J.m8 = m8;
    J.m_tiles = (p.v + 8 * m8 - 1) / (8 * m8);
    J.n_tiles = (int)((J.n_total + 127) / 128);
    J.kblocks = (p.nao + 7) / 8;
    J.out.base = Bmat + q0;
    J.out.ld_m = (long long)p.o * p.naux_ld;
    J.out.M = p.v;
    J.out.inner = pb;
    J.out.valid_inner = pb;
    J.out.stride_outer = p.naux_ld;
    J.out.n_lin_total = J.n_total;
    return SIE_OK;
}
// assign tile ranges, upload the descriptors to `d_jobs` (stream-ordered) and launch ONE grouped GEMM over all of them
int launch_jobs(std::vector<XJob>& jobs, bool packed, unsigned char* d_jobs, int num_sms, Prof& prof, int stage, cudaStream_t st) {
    if (jobs.empty()) return SIE_OK;
    long long t = 0;
    for (XJob& J : jobs) {
        J.tile_begin = (int)t;
        t += (long long)J.m_tiles * J.n_tiles;
        if (t > 0x7fffffff) return SIE_EINVAL;
    }
    SIE_CUDA(cudaMemcpyAsync(d_jobs, jobs.data(), jobs.size() * sizeof(XJob), cudaMemcpyHostToDevice, st));
    ProfSpan ps(prof, stage, st);
    return launch_xform_gemm(packed, reinterpret_cast<const XJob*>(d_jobs), (int)jobs.size(), (int)t, num_sms, st);
}

// Transform of aux rows [p0,p1) of ONE cluster into Bmat ([v][o][naux_ld]).  L points at row p0 (device, or host when
// host_L: staged through the two-buffer ring on the copy stream, one A1 launch per staged chunk).  One A1 and one A2
// launch per H sub-block otherwise.
int transform_rows(sie_dfmp2_plan_s& p, sie_dfmp2_plan_s& pipe_owner, Prof& prof, double* Bmat, const Scratch& sc, const double* dC_occ,
                   const double* dC_vir, const double* L, bool host_L, int p0, int p1, cudaStream_t st) {
    const int nao = p.nao, o = p.o, v = p.v;
    if (p.ref) {
        for (int q0 = p0; q0 < p1; q0 += p.pblk) {
            const int q1 = std::min(p1, q0 + p.pblk);
            const double* Lq = L + (size_t)(q0 - p0) * p.npair;
            if (host_L) {
                SIE_CUDA(cudaMemcpyAsync(sc.stage, Lq, (size_t)(q1 - q0) * p.npair * 8, cudaMemcpyHostToDevice, st));
                Lq = reinterpret_cast<const double*>(sc.stage);
            }
            ProfSpan ps(prof, ST_REF, st);
            SIE_TRY(ref_transform(dC_occ, dC_vir, Lq, nao, o, v, q0, q1, sc.refH, Bmat, p.naux_ld, st));
        }
        return SIE_OK;
    }
    if (host_L) {
        // the staging copies of this call must not start before earlier work on `st` that owns the workspace: ONE fork per
        // call; after that only the per-buffer ready/consumed events order the ring, so the H2D copy of chunk n+1 runs
        // under the A1 of chunk n (and the A2 of the sub-block before)
        SIE_TRY(ensure_copy_pipeline(pipe_owner));
        SIE_CUDA(cudaEventRecord(pipe_owner.ev_fork, st));
        SIE_CUDA(cudaStreamWaitEvent(pipe_owner.copy_stream, pipe_owner.ev_fork, 0));
    }
    unsigned char* arena = sc.jobs;
    int used = 0;
    std::vector<XJob> jobs(1);
    for (int q0 = p0; q0 < p1; q0 += p.pblk) {
        const int q1 = std::min(p1, q0 + p.pblk), pb = q1 - q0;
        const int step = host_L ? p.cblk : pb;
        for (int c0 = q0; c0 < q1; c0 += step) {
            const int c1 = std::min(q1, c0 + step), np = c1 - c0;
            const double* Lq = L + (size_t)(c0 - p0) * p.npair;
            int buf = 0;
            if (host_L && p.stage_full) {
                // whole-tensor staging: chunk [c0,c1) has its own place, nothing to wait for but the fork of this call
                sie_dfmp2_plan_s& po = pipe_owner;
                const size_t ci = (size_t)used;
                while (po.ev_chunk.size() <= ci) {
                    cudaEvent_t e;
                    SIE_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
                    po.ev_chunk.push_back(e);
                }
                unsigned char* dst = sc.stage + (size_t)c0 * p.npair * 8;
                SIE_CUDA(cudaMemcpyAsync(dst, Lq, (size_t)np * p.npair * 8, cudaMemcpyHostToDevice, po.copy_stream));
                SIE_CUDA(cudaEventRecord(po.ev_chunk[ci], po.copy_stream));
                SIE_CUDA(cudaStreamWaitEvent(st, po.ev_chunk[ci], 0));
                Lq = reinterpret_cast<const double*>(dst);
            } else if (host_L) {
                sie_dfmp2_plan_s& po = pipe_owner;
                buf = po.stage_turn++ & 1;
                unsigned char* dst = sc.stage + (size_t)buf * sc.stage_buf_bytes;
                SIE_CUDA(cudaStreamWaitEvent(po.copy_stream, po.ev_consumed[buf], 0));
                SIE_CUDA(cudaMemcpyAsync(dst, Lq, (size_t)np * p.npair * 8, cudaMemcpyHostToDevice, po.copy_stream));
                SIE_CUDA(cudaEventRecord(po.ev_ready[buf], po.copy_stream));
                SIE_CUDA(cudaStreamWaitEvent(st, po.ev_ready[buf], 0));
                Lq = reinterpret_cast<const double*>(dst);
            }
            if (used >= p.max_jobs) return SIE_EINVAL;  // cannot happen: max_jobs counts every chunk and sub-block
            SIE_TRY(make_a1_job(jobs[0], p, sc.CoT, Lq, np, sc.H, c0 - q0, pb));
            SIE_TRY(launch_jobs(jobs, true, arena + (size_t)used++ * sizeof(XJob), p.num_sms, prof, ST_T1, st));
            if (host_L && !p.stage_full) SIE_CUDA(cudaEventRecord(pipe_owner.ev_consumed[buf], st));
        }
        if (used >= p.max_jobs) return SIE_EINVAL;
        SIE_TRY(make_a2_job(jobs[0], p, sc.CvT, sc.H, pb, Bmat, q0));
        SIE_TRY(launch_jobs(jobs, false, arena + (size_t)used++ * sizeof(XJob), p.num_sms, prof, ST_T2, st));
    }
    return SIE_OK;
}

// transposed (K-major) copies of the coefficient matrices of one cluster
int prepare_coeffs(sie_dfmp2_plan_s& p, Prof& prof, const Scratch& sc, const double* dC_occ, const double* dC_vir,
                   cudaStream_t st) {
    if (p.ref) return SIE_OK;
    TJob tj[2] = {{dC_occ, sc.CoT, p.nao, p.o, p.nao_ld, 0}, {dC_vir, sc.CvT, p.nao, p.v, p.nao_ld, 0}};
    unsigned char* d = sc.jobs + (size_t)p.max_jobs * sizeof(XJob);
    SIE_CUDA(cudaMemcpyAsync(d, tj, sizeof tj, cudaMemcpyHostToDevice, st));
    ProfSpan ps(prof, ST_COEFF, st);
    return launch_transpose_jobs(reinterpret_cast<const TJob*>(d), 2, p.nao, std::max(p.o, p.v), st);
}

int fill_pair_cluster(const sie_dfmp2_plan_s& p, const double* Bmat, const double* de_occ, const double* de_vir, double* gpart,
                      int kp, PairCluster& d) {
    std::memset(&d, 0, sizeof d);
    const uint64_t rows = (uint64_t)p.o * p.v;  // B[a][i][P] read as a plain (v*o) x naux matrix, row = a*o + i
    SIE_TRY(make_tensor_map_3d(&d.map, Bmat, p.naux, rows, 1, (uint64_t)p.naux_ld * 8, rows * p.naux_ld * 8, 8, p.t8, 1));
    d.e_occ = de_occ;
    d.e_vir = de_vir;
    d.gpart = gpart;
    d.o = p.o;
    d.v = p.v;
    d.o8 = p.o8;
    d.ta = p.ta;
    d.kblocks = (p.naux + 7) / 8;
    d.kp = kp;
    d.t8 = p.t8;
    d.tx_bytes = 2u * 8u * (uint32_t)p.t8 * 8u;
    return SIE_OK;
}

// HOST_IO upload of a small operand.  Pinned (host-registered) memory is read by a copy kernel through its mapped device
// address, so the upload does not queue on the host-to-device copy engine behind a large staging copy of another plan;
// pageable memory takes cudaMemcpyAsync.
int stage_small(double* dst, const double* src, size_t n, cudaStream_t st) {
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, src) == cudaSuccess && at.type == cudaMemoryTypeHost && at.devicePointer)
        return launch_copy_f64(static_cast<const double*>(at.devicePointer), dst, n, st);
    (void)cudaGetLastError();
    SIE_CUDA(cudaMemcpyAsync(dst, src, n * 8, cudaMemcpyHostToDevice, st));
    return SIE_OK;
}

// the static tile list of a fused plan goes to the workspace once per workspace (first transform), not with every energy call
int upload_tiles(sie_dfmp2_plan_s& p, unsigned char* ws, cudaStream_t st) {
    if (!p.fused || p.tiles_ws == ws) return SIE_OK;
    SIE_CUDA(cudaMemcpyAsync(ws + p.off_tiles, p.tiles.data(), p.tiles.size() * sizeof(PairTile), cudaMemcpyHostToDevice, st));
    p.tiles_ws = ws;
    return SIE_OK;
}

int check_gap_host(const double* e_occ, const double* e_vir, int o, int v) {
    double mo = e_occ[0], mv = e_vir[0];
    for (int i = 1; i < o; ++i) mo = std::max(mo, e_occ[i]);
    for (int a = 1; a < v; ++a) mv = std::min(mv, e_vir[a]);
    return (mo < mv) ? SIE_OK : SIE_EGAP;  // NaN compares false -> SIE_EGAP
}

bool add_interval(std::vector<std::pair<int, int>>& cov, int p0, int p1) {
    for (auto& iv : cov)
        if (p0 < iv.second && iv.first < p1) return false;
    cov.emplace_back(p0, p1);
    return true;
}

}  // namespace

// ------------------------------------------------------------------------------------------------ C ABI
extern "C" {

int sie_dfmp2_plan(sie_dfmp2_plan_t* plan, int nao, int nocc, int nvir, int naux, int aux_block, unsigned flags,
                   size_t* workspace_bytes) {
    if (!plan || !workspace_bytes) return SIE_EINVAL;
    sie_dfmp2_plan_s* p = new (std::nothrow) sie_dfmp2_plan_s();
    if (!p) return SIE_ENOMEM;
    int rc;
    try {
        rc = plan_init(*p, nao, nocc, nvir, naux, aux_block, flags, CARVE_ALL);
    } catch (const std::bad_alloc&) {
        rc = SIE_ENOMEM;
    }
    if (rc != SIE_OK) {
        delete p;
        return rc;
    }
    p->prof.on = (flags & SIE_FLAG_PROFILE) != 0;
    *plan = p;
    *workspace_bytes = p->total;
    return SIE_OK;
}

int sie_dfmp2_transform(sie_dfmp2_plan_t plan, void* workspace, const double* C_occ, const double* C_vir,
                        const double* L_packed_block, int p0, int p1, void* cuda_stream) {
    if (!plan || !workspace || !C_occ || !C_vir || !L_packed_block) return SIE_EINVAL;
    sie_dfmp2_plan_s& p = *plan;
    if (p0 < 0 || p1 > p.naux || p0 >= p1) return SIE_EINVAL;
    if (reinterpret_cast<uintptr_t>(workspace) & 255) return SIE_EINVAL;
    SIE_TRY(check_device());
    // B of the rows covered so far lives in the workspace they were transformed into: a different workspace mid-way
    // would leave rows missing (sie_dfmp2_plan_reset starts over)
    if (!p.covered.empty() && p.c_ready_ws != workspace) return SIE_ESTATE;
    for (auto& iv : p.covered)
        if (p0 < iv.second && iv.first < p1) return SIE_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    unsigned char* ws = static_cast<unsigned char*>(workspace);
    const bool host = p.flags & SIE_FLAG_HOST_IO;
    Scratch sc{};
    sc.CoT = reinterpret_cast<double*>(ws + p.off_CoT);
    sc.CvT = reinterpret_cast<double*>(ws + p.off_CvT);
    sc.H = reinterpret_cast<double*>(ws + p.off_H);
    sc.jobs = ws + p.off_jobs;
    sc.refH = reinterpret_cast<double*>(ws + p.off_refH);
    sc.stage = ws + p.off_stage;
    sc.stage_buf_bytes = p.stage_buf_bytes;
    if (p.c_ready_ws != workspace || p.covered.empty()) {
        const double *dCo = C_occ, *dCv = C_vir;
        if (host) {
            double* io = reinterpret_cast<double*>(ws + p.off_io);
            SIE_CUDA(cudaMemcpyAsync(io + p.io_Cocc, C_occ, (size_t)p.nao * p.o * 8, cudaMemcpyHostToDevice, st));
            SIE_CUDA(cudaMemcpyAsync(io + p.io_Cvir, C_vir, (size_t)p.nao * p.v * 8, cudaMemcpyHostToDevice, st));
            dCo = io + p.io_Cocc;
            dCv = io + p.io_Cvir;
        }
        SIE_TRY(prepare_coeffs(p, p.prof, sc, dCo, dCv, st));
        SIE_TRY(upload_tiles(p, ws, st));
        p.dC_occ = dCo;
        p.dC_vir = dCv;
        p.c_ready_ws = workspace;
    }
    SIE_TRY(transform_rows(p, p, p.prof, reinterpret_cast<double*>(ws + p.off_B), sc, p.dC_occ, p.dC_vir, L_packed_block, host, p0, p1, st));
    add_interval(p.covered, p0, p1);
    p.covered_rows += p1 - p0;
    return SIE_OK;
}

static int energy_impl(sie_dfmp2_plan_t plan, void* workspace, const double* e_occ, const double* e_vir, const double* P_frag,
                       double* E_out, double* G_out, void* cuda_stream, int mode) {
    if (!plan || !workspace || !e_occ || !e_vir || (!E_out && mode == 0)) return SIE_EINVAL;
    sie_dfmp2_plan_s& p = *plan;
    if (p.covered_rows != p.naux || p.c_ready_ws != workspace) return SIE_ESTATE;
    SIE_TRY(check_device());
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    unsigned char* ws = static_cast<unsigned char*>(workspace);
    const bool host = p.flags & SIE_FLAG_HOST_IO;
    const int o = p.o, v = p.v;

    const double *de_occ = e_occ, *de_vir = e_vir, *dP = P_frag;
    double *dE = E_out, *dG = G_out;
    if (!dE) dE = reinterpret_cast<double*>(ws + p.off_rc + 128);  // mode 1 without a trace output: spare bytes behind the descriptor
    double* io = reinterpret_cast<double*>(ws + p.off_io);
    if (host) {
        if (p.flags & SIE_FLAG_VALIDATE) SIE_TRY(check_gap_host(e_occ, e_vir, o, v));
        SIE_TRY(stage_small(io + p.io_eo, e_occ, (size_t)o, st));
        SIE_TRY(stage_small(io + p.io_ev, e_vir, (size_t)v, st));
        de_occ = io + p.io_eo;
        de_vir = io + p.io_ev;
        if (P_frag) {
            SIE_TRY(stage_small(io + p.io_P, P_frag, (size_t)o * o, st));
            dP = io + p.io_P;
        }
        dE = io + p.io_E;
        dG = G_out ? io + p.io_G : nullptr;
    } else if (p.flags & SIE_FLAG_VALIDATE) {
        std::vector<double> he(o + v);
        SIE_CUDA(cudaMemcpyAsync(he.data(), e_occ, (size_t)o * 8, cudaMemcpyDeviceToHost, st));
        SIE_CUDA(cudaMemcpyAsync(he.data() + o, e_vir, (size_t)v * 8, cudaMemcpyDeviceToHost, st));
        SIE_CUDA(cudaStreamSynchronize(st));
        SIE_TRY(check_gap_host(he.data(), he.data() + o, o, v));
    }

    const double* Bmat = reinterpret_cast<const double*>(ws + p.off_B);
    ReduceCluster rc{};
    rc.P = dP;
    rc.E_out = dE;
    rc.G_out = dG;
    rc.o = o;
    rc.mode = mode;
    if (p.ref) {
        double* G = reinterpret_cast<double*>(ws + p.off_refG);
        {
            ProfSpan ps(p.prof, ST_REF, st);
            SIE_TRY(ref_pair(Bmat, o, v, p.naux, p.naux_ld, de_occ, de_vir, reinterpret_cast<double*>(ws + p.off_refVj), G, mode, st));
        }
        rc.gpart = G;
        rc.o8 = o;
        rc.nslots = 1;
    } else if (p.general || mode == 2) {
        // any-size route (general.cu): nocc > 128, and the virtual 1-RDM block at every size
        if (!p.has_gen) return SIE_ESTATE;  // gamma_vir needs a plan created with SIE_FLAG_RDM_VIR
        double* slots = reinterpret_cast<double*>(ws + p.off_gslots);
        int nslots = 0;
        {
            ProfSpan ps(p.prof, ST_PAIR, st);
            SIE_TRY(general_pair(p.gen, Bmat, o, v, p.naux, p.naux_ld, de_occ, de_vir, mode, ws + p.off_gen, slots, &nslots, p.num_sms, st));
        }
        rc.gpart = slots;
        rc.o = mode == 2 ? v : o;
        rc.o8 = rc.o;
        rc.nslots = nslots;
    } else {
        double* gpart = reinterpret_cast<double*>(ws + p.off_gpart);
        PairCluster pc;
        SIE_TRY(fill_pair_cluster(p, Bmat, de_occ, de_vir, gpart, p.kp, pc));
        // one cluster: all tiles cost the same, keep the CTAs in K-lockstep for L2.  Energy mode only: in the amplitude mode
        // (gamma_occ) the gate costs 5 % at config 3 (2538 -> 2668 ms) because its pre-pass shifts the CTAs' phases
        pc.gate = mode == 0 ? 1 : 0;
        pc.mode = mode;
        SIE_TRY(launch_poke(&pc, sizeof pc, ws + p.off_desc, st));
        SIE_TRY(upload_tiles(p, ws, st));
        SIE_CUDA(cudaMemsetAsync(ws + p.off_tiles + p.tiles.size() * sizeof(PairTile), 0, 256, st));
        SIE_CUDA(cudaMemsetAsync(gpart, 0, (size_t)p.ncta * p.kp * p.o8 * p.o8 * 8, st));
        {
            ProfSpan ps(p.prof, ST_PAIR, st);
            SIE_TRY(launch_pair(reinterpret_cast<const PairCluster*>(ws + p.off_desc),
                                reinterpret_cast<const PairTile*>(ws + p.off_tiles), (int)p.tiles.size(), p.ncta, p.t8,
                                (mode == 0 && pair_small_strip(o, pair_producer_warp(p.t8) != 0)) ? 3 : mode, pair_producer_warp(p.t8), st));
        }
        rc.gpart = gpart;
        rc.o8 = p.o8;
        rc.nslots = p.ncta * p.kp;
    }
    SIE_TRY(launch_poke(&rc, sizeof rc, ws + p.off_rc, st));
    {
        ProfSpan ps(p.prof, ST_REDUCE, st);
        SIE_TRY(launch_reduce(reinterpret_cast<const ReduceCluster*>(ws + p.off_rc), 1, st));
    }
    if (host) {
        if (E_out) SIE_CUDA(cudaMemcpyAsync(E_out, dE, 8, cudaMemcpyDeviceToHost, st));
        if (G_out) SIE_CUDA(cudaMemcpyAsync(G_out, dG, (size_t)rc.o * rc.o * 8, cudaMemcpyDeviceToHost, st));
        SIE_CUDA(cudaStreamSynchronize(st));
    }
    return SIE_OK;
}

int sie_dfmp2_energy(sie_dfmp2_plan_t plan, void* workspace, const double* e_occ, const double* e_vir, const double* P_frag,
                     double* E_out, double* G_out, void* cuda_stream) {
    return energy_impl(plan, workspace, e_occ, e_vir, P_frag, E_out, G_out, cuda_stream, 0);
}

int sie_dfmp2_rdm_occ(sie_dfmp2_plan_t plan, void* workspace, const double* e_occ, const double* e_vir, double* gamma_out,
                      double* trace_out, void* cuda_stream) {
    if (!gamma_out) return SIE_EINVAL;
    return energy_impl(plan, workspace, e_occ, e_vir, nullptr, trace_out, gamma_out, cuda_stream, 1);
}

int sie_dfmp2_energy_lowrank(sie_dfmp2_plan_t plan, void* workspace, const double* e_occ, const double* e_vir, const double* Q, int r,
                             double* E_out, void* cuda_stream) {
    if (!plan || !workspace || !e_occ || !e_vir || !Q || !E_out || r < 1 || r > plan->o) return SIE_EINVAL;
    sie_dfmp2_plan_s& p = *plan;
    if (p.covered_rows != p.naux || p.c_ready_ws != workspace) return SIE_ESTATE;
    if (!p.fused) return SIE_EUNSUPPORTED;  // general / reference routes: form P = Q Q^T and call sie_dfmp2_energy
    SIE_TRY(check_device());
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    unsigned char* ws = static_cast<unsigned char*>(workspace);
    const bool host = p.flags & SIE_FLAG_HOST_IO;
    const int o = p.o, v = p.v;
    const double *de_occ = e_occ, *de_vir = e_vir, *dQ = Q;
    double* dE = E_out;
    double* io = reinterpret_cast<double*>(ws + p.off_io);
    if (host) {
        if (p.flags & SIE_FLAG_VALIDATE) SIE_TRY(check_gap_host(e_occ, e_vir, o, v));
        SIE_TRY(stage_small(io + p.io_eo, e_occ, (size_t)o, st));
        SIE_TRY(stage_small(io + p.io_ev, e_vir, (size_t)v, st));
        SIE_TRY(stage_small(io + p.io_P, Q, (size_t)o * r, st));  // r <= o: fits the P slot
        de_occ = io + p.io_eo;
        de_vir = io + p.io_ev;
        dQ = io + p.io_P;
        dE = io + p.io_E;
    } else if (p.flags & SIE_FLAG_VALIDATE) {
        std::vector<double> he(o + v);
        SIE_CUDA(cudaMemcpyAsync(he.data(), e_occ, (size_t)o * 8, cudaMemcpyDeviceToHost, st));
        SIE_CUDA(cudaMemcpyAsync(he.data() + o, e_vir, (size_t)v * 8, cudaMemcpyDeviceToHost, st));
        SIE_CUDA(cudaStreamSynchronize(st));
        SIE_TRY(check_gap_host(he.data(), he.data() + o, o, v));
    }
    const double* Bmat = reinterpret_cast<const double*>(ws + p.off_B);
    double* Qt = reinterpret_cast<double*>(ws + p.off_Qt);
    double* Pbuf = Qt + (size_t)32 * p.o8;
    double* gpart = reinterpret_cast<double*>(ws + p.off_gpart);
    const int r8 = (r + 7) / 8;
    const bool lowrank = r8 <= 4;
    ReduceCluster rc{};
    rc.E_out = dE;
    PairCluster pc;
    SIE_TRY(fill_pair_cluster(p, Bmat, de_occ, de_vir, gpart, p.kp, pc));
    pc.gate = 1;
    SIE_TRY(launch_lowrank_prep(dQ, o, r, lowrank ? Qt : nullptr, p.o8, r8, lowrank ? nullptr : Pbuf, st));
    if (lowrank) {  // contract with Q^T first: per-warp partial energies, no G
        pc.mode = 2;
        pc.Qt = Qt;
        pc.r8 = r8;
        pc.ldq = p.o8;
        SIE_CUDA(cudaMemsetAsync(gpart, 0, (size_t)p.ncta * pair_geom().ncons * 8, st));
        rc.o = 1;
        rc.o8 = 1;
        rc.nslots = p.ncta * pair_geom().ncons;
    } else {        // rank above 32: the o x o x o epilogue is the cheaper one; P = Q Q^T through the G path
        pc.mode = 0;
        SIE_CUDA(cudaMemsetAsync(gpart, 0, (size_t)p.ncta * p.kp * p.o8 * p.o8 * 8, st));
        rc.P = Pbuf;
        rc.o = o;
        rc.o8 = p.o8;
        rc.nslots = p.ncta * p.kp;
    }
    rc.gpart = gpart;
    SIE_TRY(launch_poke(&pc, sizeof pc, ws + p.off_desc, st));
    SIE_TRY(upload_tiles(p, ws, st));
    SIE_CUDA(cudaMemsetAsync(ws + p.off_tiles + p.tiles.size() * sizeof(PairTile), 0, 256, st));
    {
        ProfSpan ps(p.prof, ST_PAIR, st);
        SIE_TRY(launch_pair(reinterpret_cast<const PairCluster*>(ws + p.off_desc), reinterpret_cast<const PairTile*>(ws + p.off_tiles),
                            (int)p.tiles.size(), p.ncta, p.t8, pc.mode, pair_producer_warp(p.t8), st));
    }
    SIE_TRY(launch_poke(&rc, sizeof rc, ws + p.off_rc, st));
    {
        ProfSpan ps(p.prof, ST_REDUCE, st);
        SIE_TRY(launch_reduce(reinterpret_cast<const ReduceCluster*>(ws + p.off_rc), 1, st));
    }
    if (host) {
        SIE_CUDA(cudaMemcpyAsync(E_out, dE, 8, cudaMemcpyDeviceToHost, st));
        SIE_CUDA(cudaStreamSynchronize(st));
    }
    return SIE_OK;
}

int sie_dfmp2_rdm_vir(sie_dfmp2_plan_t plan, void* workspace, const double* e_occ, const double* e_vir, double* gamma_out,
                      double* trace_out, void* cuda_stream) {
    if (!gamma_out) return SIE_EINVAL;
    if (plan && plan->ref) return SIE_EUNSUPPORTED;  // the reference kernels have no virtual-block mode
    return energy_impl(plan, workspace, e_occ, e_vir, nullptr, trace_out, gamma_out, cuda_stream, 2);
}

int sie_dfmp2_batch(int ncluster, const sie_dfmp2_cluster_t* clusters, void* workspace, size_t workspace_bytes, size_t* needed,
                    unsigned flags, void* cuda_stream) {
    if (ncluster < 0 || (ncluster > 0 && !clusters)) return SIE_EINVAL;
    if (flags & ~(SIE_FLAG_VALIDATE | SIE_FLAG_REFERENCE | SIE_FLAG_HOST_IO | SIE_FLAG_PROFILE | SIE_FLAG_RDM_OCC)) return SIE_EINVAL;
    const bool host = flags & SIE_FLAG_HOST_IO;
    const int mode = (flags & SIE_FLAG_RDM_OCC) ? 1 : 0;
    const bool query = (workspace == nullptr || workspace_bytes == 0);
    if (query && !needed) return SIE_EINVAL;
    if (ncluster == 0) {  // nothing to schedule: no workspace, no launch
        if (needed) *needed = 0;
        return SIE_OK;
    }
    try {
        // ---- per-cluster plans.  Device pointers: every fused-path cluster owns B, partial-G slots, coefficient copies and
        //      an H sub-block, so ONE grouped launch per transform stage serves all clusters.  Host pointers: the packed
        //      integrals go through one staging ring, cluster by cluster, with shared scratch sized for the largest cluster.
        std::vector<sie_dfmp2_plan_s> plans(ncluster);
        Carver c;
        std::vector<size_t> off_cl(ncluster), off_io(ncluster);
        // Clusters of ONE system share their three-index integrals (the SIE access pattern: every cluster is a
        // different orbital set C over the same (P|mu nu)): members of a batch that pass the same L_packed pointer with the
        // same nao and naux are transformed together — their C_occ columns are stacked into one A1 GEMM, so (P|mu nu) is
        // read once for all of them instead of once per cluster.  (Device pointers only.  The workspace layout depends on
        // the grouping, so a size query must be made with the same descriptors, pointers included, as the call.)
        struct SharedGroup {
            std::vector<int> members;
            std::vector<int> row0;  // first stacked occupied row of each member
            int o_sum = 0, pblk = 0;
            size_t off_CoT = 0, off_H = 0;
        };
        std::vector<SharedGroup> groups;
        std::vector<int> group_of(ncluster, -1);
        std::vector<size_t> off_CvT_shared(ncluster, 0);
        if (!host && !(flags & SIE_FLAG_REFERENCE)) {
            for (int k = 0; k < ncluster; ++k) {
                if (!clusters[k].L_packed || group_of[k] >= 0) continue;
                SharedGroup g;
                for (int m = k; m < ncluster; ++m)
                    if (group_of[m] < 0 && clusters[m].L_packed == clusters[k].L_packed && clusters[m].nao == clusters[k].nao &&
                        clusters[m].naux == clusters[k].naux)
                        g.members.push_back(m);
                if (g.members.size() < 2) continue;
                for (int m : g.members) group_of[m] = (int)groups.size();
                groups.push_back(g);
            }
        }
        size_t max_CoT = 0, max_CvT = 0, max_H = 0, max_refH = 0, max_refVj = 0, max_stage = 0, ntiles_total = 0, max_jobs1 = 0, group_jobs = 0, max_gen = 0;
        int nfused = 0;
        for (int k = 0; k < ncluster; ++k) {
            const sie_dfmp2_cluster_t& cl = clusters[k];
            if (!query && (!cl.C_occ || !cl.C_vir || !cl.L_packed || !cl.e_occ || !cl.e_vir || !cl.E_out)) return SIE_EINVAL;
            sie_dfmp2_plan_s& p = plans[k];
            SIE_TRY(plan_init(p, cl.nao, cl.nocc, cl.nvir, cl.naux, 0, flags & ~(SIE_FLAG_HOST_IO | SIE_FLAG_PROFILE | SIE_FLAG_RDM_OCC),
                              (host || group_of[k] >= 0) ? CARVE_NONE : CARVE_MEMBER));
            off_cl[k] = c.take(p.total);
            if (group_of[k] >= 0) off_CvT_shared[k] = c.take((size_t)p.v * p.nao_ld * 8);
            if (!p.ref) {
                ++nfused;
                max_CoT = std::max(max_CoT, (size_t)p.o * p.nao_ld * 8);
                max_CvT = std::max(max_CvT, (size_t)p.v * p.nao_ld * 8);
                max_H = std::max(max_H, (size_t)p.o * p.pblk * p.nao_ld * 8);
                max_jobs1 = std::max(max_jobs1, (size_t)p.max_jobs);
                if (group_of[k] < 0) group_jobs += 2 * (size_t)((p.naux + p.pblk - 1) / p.pblk);
                ntiles_total += p.tiles.size();
            } else {
                max_refH = std::max(max_refH, (size_t)p.pblk * p.o * p.nao * 8);
                max_refVj = std::max(max_refVj, ref_vj_bytes(p.o, p.v));
            }
            if (p.has_gen) max_gen = std::max(max_gen, general_scratch_bytes(p.gen, p.o));
            max_stage = std::max(max_stage, align_up((size_t)p.cblk * p.npair * 8, 256));
            if (host) {
                size_t d = (size_t)p.nao * p.o + (size_t)p.nao * p.v + p.o + p.v + 2 * (size_t)p.o * p.o + 2;
                off_io[k] = c.take(d * 8);
            }
        }
        for (SharedGroup& g : groups) {
            const sie_dfmp2_plan_s& p0 = plans[g.members[0]];
            for (int m : g.members) {
                g.row0.push_back(g.o_sum);
                g.o_sum += plans[m].o;
            }
            const size_t per_p = (size_t)g.o_sum * p0.nao_ld * 8;
            long long pb = std::max<long long>(8, (long long)(((size_t)2 << 30) / per_p));
            pb = std::min<long long>(pb, (long long)0x7fffffff / std::max(p0.nao, g.o_sum) - 1);
            if (pb < p0.naux) pb = std::max<long long>(8, pb / 8 * 8);
            g.pblk = (int)std::min<long long>(pb, p0.naux);
            g.off_CoT = c.take((size_t)g.o_sum * p0.nao_ld * 8);
            g.off_H = c.take((size_t)g.o_sum * g.pblk * p0.nao_ld * 8);
            group_jobs += (size_t)((p0.naux + g.pblk - 1) / g.pblk) * (1 + g.members.size());
        }
        size_t off_CoT = 0, off_CvT = 0, off_H = 0;
        if (host) {
            off_CoT = c.take(max_CoT);
            off_CvT = c.take(max_CvT);
            off_H = c.take(max_H);
        }
        const size_t off_refH = c.take(max_refH);
        const size_t off_refVj = c.take(max_refVj);
        const size_t off_gen = c.take(max_gen);
        const size_t off_stage = host ? c.take(2 * max_stage) : 0;
        const size_t njobs_arena = host ? max_jobs1 : group_jobs;
        const size_t off_jobs = c.take(njobs_arena * sizeof(XJob) + 2 * (size_t)std::max(1, ncluster) * sizeof(TJob));
        const size_t off_desc = c.take((size_t)std::max(1, ncluster) * sizeof(PairCluster));
        const size_t off_tiles = c.take(std::max<size_t>(1, ntiles_total) * sizeof(PairTile) + 256);
        const size_t off_rc = c.take((size_t)std::max(1, ncluster) * sizeof(ReduceCluster));
        const size_t total = c.off;
        if (needed) *needed = total;
        if (query) return SIE_OK;
        if (workspace_bytes < total) return SIE_ENOMEM;
        if (reinterpret_cast<uintptr_t>(workspace) & 255) return SIE_EINVAL;
        if (ncluster == 0) return SIE_OK;
        SIE_TRY(check_device());

        cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
        unsigned char* ws = static_cast<unsigned char*>(workspace);
        Prof& prof = g_batch_prof;
        prof.reset();
        prof.on = (flags & SIE_FLAG_PROFILE) != 0;
        sie_dfmp2_plan_s pipe;  // owns the HOST_IO copy stream/events of this call
        struct PipeGuard {
            sie_dfmp2_plan_s& p;
            ~PipeGuard() {
                if (p.copy_stream) {
                    cudaStreamSynchronize(p.copy_stream);
                    for (int i = 0; i < 2; ++i) {
                        cudaEventDestroy(p.ev_ready[i]);
                        cudaEventDestroy(p.ev_consumed[i]);
                    }
                    cudaEventDestroy(p.ev_fork);
                    cudaStreamDestroy(p.copy_stream);
                    p.copy_stream = nullptr;
                }
            }
        } guard{pipe};

        std::vector<PairCluster> descs(ncluster);
        std::vector<ReduceCluster> rcs(ncluster);
        std::vector<const double*> de_occ(ncluster), de_vir(ncluster), dCo(ncluster), dCv(ncluster);
        std::vector<double*> dE(ncluster), dG(ncluster);
        // ---- stage 0: per-cluster pointers (host pointers: small operands uploaded; VALIDATE: gap check)
        for (int k = 0; k < ncluster; ++k) {
            const sie_dfmp2_cluster_t& cl = clusters[k];
            sie_dfmp2_plan_s& p = plans[k];
            const double* dP = cl.P_frag;
            dCo[k] = cl.C_occ;
            dCv[k] = cl.C_vir;
            de_occ[k] = cl.e_occ;
            de_vir[k] = cl.e_vir;
            dE[k] = cl.E_out;
            dG[k] = cl.G_out;
            if (host) {
                if (flags & SIE_FLAG_VALIDATE) SIE_TRY(check_gap_host(cl.e_occ, cl.e_vir, p.o, p.v));
                double* io = reinterpret_cast<double*>(ws + off_io[k]);
                size_t d = 0;
                auto up = [&](const double* src, size_t n) -> const double* {
                    double* dst = io + d;
                    d += n;
                    return cudaMemcpyAsync(dst, src, n * 8, cudaMemcpyHostToDevice, st) == cudaSuccess ? dst : nullptr;
                };
                dCo[k] = up(cl.C_occ, (size_t)p.nao * p.o);
                dCv[k] = up(cl.C_vir, (size_t)p.nao * p.v);
                de_occ[k] = up(cl.e_occ, p.o);
                de_vir[k] = up(cl.e_vir, p.v);
                if (cl.P_frag) dP = up(cl.P_frag, (size_t)p.o * p.o);
                if (!dCo[k] || !dCv[k] || !de_occ[k] || !de_vir[k] || (cl.P_frag && !dP)) return set_cuda_error(cudaGetLastError());
                dE[k] = io + d;
                d += 2;
                dG[k] = cl.G_out ? io + d : nullptr;
            } else if (flags & SIE_FLAG_VALIDATE) {
                std::vector<double> he(p.o + p.v);
                SIE_CUDA(cudaMemcpyAsync(he.data(), cl.e_occ, (size_t)p.o * 8, cudaMemcpyDeviceToHost, st));
                SIE_CUDA(cudaMemcpyAsync(he.data() + p.o, cl.e_vir, (size_t)p.v * 8, cudaMemcpyDeviceToHost, st));
                SIE_CUDA(cudaStreamSynchronize(st));
                SIE_TRY(check_gap_host(he.data(), he.data() + p.o, p.o, p.v));
            }
            rcs[k] = ReduceCluster{};
            rcs[k].P = dP;
            rcs[k].E_out = dE[k];
            rcs[k].G_out = dG[k];
            rcs[k].o = p.o;
            rcs[k].mode = mode;
            if (mode) rcs[k].P = nullptr;
        }
        // ---- stage 1: transforms (A1, A2)
        unsigned char* arena = ws + off_jobs;
        if (host) {
            Scratch sc{};
            sc.CoT = reinterpret_cast<double*>(ws + off_CoT);
            sc.CvT = reinterpret_cast<double*>(ws + off_CvT);
            sc.H = reinterpret_cast<double*>(ws + off_H);
            sc.refH = reinterpret_cast<double*>(ws + off_refH);
            sc.stage = ws + off_stage;
            sc.stage_buf_bytes = max_stage;
            for (int k = 0; k < ncluster; ++k) {
                sie_dfmp2_plan_s& p = plans[k];
                // this cluster's descriptors: max_jobs XJobs, then its two TJobs (prepare_coeffs expects them right behind)
                sc.jobs = arena + (max_jobs1 - (size_t)p.max_jobs) * sizeof(XJob);
                SIE_TRY(prepare_coeffs(p, prof, sc, dCo[k], dCv[k], st));
                SIE_TRY(transform_rows(p, pipe, prof, reinterpret_cast<double*>(ws + off_cl[k] + p.off_B), sc, dCo[k], dCv[k],
                                       clusters[k].L_packed, true, 0, p.naux, st));
            }
        } else {
            // one transpose launch, then per round r (the r-th H sub-block of every cluster / shared group) ONE A1 and ONE A2 launch
            std::vector<TJob> tj;
            int max_rows = 1, max_cols = 1, rounds = 0;
            std::vector<double*> CvT(ncluster, nullptr);
            for (int k = 0; k < ncluster; ++k) {
                sie_dfmp2_plan_s& p = plans[k];
                if (p.ref) continue;
                unsigned char* wk = ws + off_cl[k];
                double* CoT;
                if (group_of[k] >= 0) {
                    const SharedGroup& g = groups[group_of[k]];
                    const int idx = (int)(std::find(g.members.begin(), g.members.end(), k) - g.members.begin());
                    CoT = reinterpret_cast<double*>(ws + g.off_CoT) + (size_t)g.row0[idx] * p.nao_ld;
                    CvT[k] = reinterpret_cast<double*>(ws + off_CvT_shared[k]);
                    rounds = std::max(rounds, (p.naux + g.pblk - 1) / g.pblk);
                } else {
                    CoT = reinterpret_cast<double*>(wk + p.off_CoT);
                    CvT[k] = reinterpret_cast<double*>(wk + p.off_CvT);
                    rounds = std::max(rounds, (p.naux + p.pblk - 1) / p.pblk);
                }
                tj.push_back(TJob{dCo[k], CoT, p.nao, p.o, p.nao_ld, 0});
                tj.push_back(TJob{dCv[k], CvT[k], p.nao, p.v, p.nao_ld, 0});
                max_rows = std::max(max_rows, p.nao);
                max_cols = std::max(max_cols, std::max(p.o, p.v));
            }
            if (!tj.empty()) {
                unsigned char* d = arena + njobs_arena * sizeof(XJob);
                SIE_CUDA(cudaMemcpyAsync(d, tj.data(), tj.size() * sizeof(TJob), cudaMemcpyHostToDevice, st));
                ProfSpan ps(prof, ST_COEFF, st);
                SIE_TRY(launch_transpose_jobs(reinterpret_cast<const TJob*>(d), (int)tj.size(), max_rows, max_cols, st));
            }
            size_t used = 0;
            std::vector<XJob> j1, j2;
            for (int r = 0; r < rounds; ++r) {
                j1.clear();
                j2.clear();
                XJob J;
                for (int k = 0; k < ncluster; ++k) {  // clusters with private integrals
                    sie_dfmp2_plan_s& p = plans[k];
                    if (p.ref || group_of[k] >= 0) continue;
                    const int q0 = r * p.pblk;
                    if (q0 >= p.naux) continue;
                    const int pb = std::min(p.pblk, p.naux - q0);
                    unsigned char* wk = ws + off_cl[k];
                    double* H = reinterpret_cast<double*>(wk + p.off_H);
                    SIE_TRY(make_a1_job(J, p, reinterpret_cast<const double*>(wk + p.off_CoT), clusters[k].L_packed + (size_t)q0 * p.npair, pb,
                                        H, 0, pb));
                    j1.push_back(J);
                    SIE_TRY(make_a2_job(J, p, CvT[k], H, pb, reinterpret_cast<double*>(wk + p.off_B), q0));
                    j2.push_back(J);
                }
                for (const SharedGroup& g : groups) {  // shared integrals: one A1 job over the stacked occupied columns
                    const int k0 = g.members[0];
                    sie_dfmp2_plan_s pg = plans[k0];  // a copy that stands for the stacked cluster (sizes only)
                    pg.o = g.o_sum;
                    const int q0 = r * g.pblk;
                    if (q0 >= pg.naux) continue;
                    const int pb = std::min(g.pblk, pg.naux - q0);
                    double* H = reinterpret_cast<double*>(ws + g.off_H);
                    SIE_TRY(make_a1_job(J, pg, reinterpret_cast<const double*>(ws + g.off_CoT), clusters[k0].L_packed + (size_t)q0 * pg.npair,
                                        pb, H, 0, pb));
                    j1.push_back(J);
                    for (size_t m = 0; m < g.members.size(); ++m) {
                        const int k = g.members[m];
                        sie_dfmp2_plan_s& p = plans[k];
                        // member rows [row0, row0 + o) of H[i][P][nu] are one contiguous slice
                        SIE_TRY(make_a2_job(J, p, CvT[k], H + (size_t)g.row0[m] * pb * p.nao_ld, pb,
                                            reinterpret_cast<double*>(ws + off_cl[k] + p.off_B), q0));
                        j2.push_back(J);
                    }
                }
                if (used + j1.size() + j2.size() > njobs_arena) return SIE_EINVAL;  // cannot happen: counted above
                SIE_TRY(launch_jobs(j1, true, arena + used * sizeof(XJob), plans[0].num_sms, prof, ST_T1, st));
                used += j1.size();
                SIE_TRY(launch_jobs(j2, false, arena + used * sizeof(XJob), plans[0].num_sms, prof, ST_T2, st));
                used += j2.size();
            }
            for (int k = 0; k < ncluster; ++k) {  // reference-path clusters: simple kernels, one cluster at a time
                sie_dfmp2_plan_s& p = plans[k];
                if (!p.ref) continue;
                Scratch sc{};
                sc.refH = reinterpret_cast<double*>(ws + off_refH);
                SIE_TRY(transform_rows(p, pipe, prof, reinterpret_cast<double*>(ws + off_cl[k] + p.off_B), sc, dCo[k], dCv[k],
                                       clusters[k].L_packed, false, 0, p.naux, st));
            }
        }
        // ---- stage 2: one persistent pair launch over all (cluster, tile) items, most expensive tiles first
        std::vector<int> order;
        for (int k = 0; k < ncluster; ++k)
            if (plans[k].fused) order.push_back(k);
        std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return plans[a].tile_cost > plans[b].tile_cost; });
        const int ncta = (int)std::min<size_t>((size_t)plans[0].num_sms, std::max<size_t>(1, ntiles_total));
        std::vector<PairTile> tiles;
        tiles.reserve(ntiles_total);
        int tmax = 8;
        for (int k : order) tmax = std::max(tmax, plans[k].t8);
        for (int k : order) {
            sie_dfmp2_plan_s& p = plans[k];
            unsigned char* wk = ws + off_cl[k];
            double* gpart = reinterpret_cast<double*>(wk + p.off_gpart);
            SIE_TRY(fill_pair_cluster(p, reinterpret_cast<const double*>(wk + p.off_B), de_occ[k], de_vir[k], gpart, p.kp, descs[k]));
            SIE_CUDA(cudaMemsetAsync(gpart, 0, (size_t)ncta * p.kp * p.o8 * p.o8 * 8, st));
            for (PairTile t : p.tiles) {
                t.cluster = k;
                tiles.push_back(t);
            }
            rcs[k].gpart = gpart;
            rcs[k].o8 = p.o8;
            rcs[k].nslots = ncta * p.kp;
        }
        if (!tiles.empty()) {
            SIE_CUDA(cudaMemcpyAsync(ws + off_desc, descs.data(), descs.size() * sizeof(PairCluster), cudaMemcpyHostToDevice, st));
            SIE_CUDA(cudaMemcpyAsync(ws + off_tiles, tiles.data(), tiles.size() * sizeof(PairTile), cudaMemcpyHostToDevice, st));
            SIE_CUDA(cudaMemsetAsync(ws + off_tiles + tiles.size() * sizeof(PairTile), 0, 256, st));
            ProfSpan ps(prof, ST_PAIR, st);
            // the polling producer (sie_internal.h) as soon as a third of the batch's tile work has a warp with time to spare
            // (config 2: 49 % of the work, 480.1 -> 470.8 ms; a launch of even 128-row tiles alone loses 5 % with it)
            double cost_uneven = 0.0, cost_even = 0.0;
            for (int k : order) (pair_producer_warp(plans[k].t8) ? cost_uneven : cost_even) += plans[k].tile_cost * (double)plans[k].tiles.size();
            const int pw = 3.0 * cost_uneven >= cost_uneven + cost_even ? 12 : 0;
            bool any_small = false;
            for (int k : order) any_small = any_small || pair_small_strip(plans[k].o, pw != 0);
            SIE_TRY(launch_pair(reinterpret_cast<const PairCluster*>(ws + off_desc), reinterpret_cast<const PairTile*>(ws + off_tiles),
                                (int)tiles.size(), ncta, tmax, (mode == 0 && any_small) ? 3 : mode, pw, st));
        }
        // clusters with nocc > 128: the any-size slab/Gram route, one cluster at a time on shared scratch
        for (int k = 0; k < ncluster; ++k) {
            sie_dfmp2_plan_s& p = plans[k];
            if (!p.general) continue;
            unsigned char* wk = ws + off_cl[k];
            double* slots = reinterpret_cast<double*>(wk + p.off_gslots);
            int nslots = 0;
            {
                ProfSpan ps(prof, ST_PAIR, st);
                SIE_TRY(general_pair(p.gen, reinterpret_cast<const double*>(wk + p.off_B), p.o, p.v, p.naux, p.naux_ld, de_occ[k], de_vir[k],
                                     mode, ws + off_gen, slots, &nslots, p.num_sms, st));
            }
            rcs[k].gpart = slots;
            rcs[k].o8 = p.o;
            rcs[k].nslots = nslots;
        }
        // reference-path clusters (SIE_FLAG_REFERENCE): per-j kernels, one cluster at a time
        for (int k = 0; k < ncluster; ++k) {
            sie_dfmp2_plan_s& p = plans[k];
            if (!p.ref) continue;
            unsigned char* wk = ws + off_cl[k];
            double* G = reinterpret_cast<double*>(wk + p.off_refG);
            {
                ProfSpan ps(prof, ST_REF, st);
                SIE_TRY(ref_pair(reinterpret_cast<const double*>(wk + p.off_B), p.o, p.v, p.naux, p.naux_ld, de_occ[k], de_vir[k],
                                 reinterpret_cast<double*>(ws + off_refVj), G, mode, st));
            }
            rcs[k].gpart = G;
            rcs[k].o8 = p.o;
            rcs[k].nslots = 1;
        }
        SIE_CUDA(cudaMemcpyAsync(ws + off_rc, rcs.data(), rcs.size() * sizeof(ReduceCluster), cudaMemcpyHostToDevice, st));
        {
            ProfSpan ps(prof, ST_REDUCE, st);
            SIE_TRY(launch_reduce(reinterpret_cast<const ReduceCluster*>(ws + off_rc), ncluster, st));
        }
        if (host) {
            for (int k = 0; k < ncluster; ++k) {
                SIE_CUDA(cudaMemcpyAsync(clusters[k].E_out, dE[k], 8, cudaMemcpyDeviceToHost, st));
                if (clusters[k].G_out)
                    SIE_CUDA(cudaMemcpyAsync(clusters[k].G_out, dG[k], (size_t)plans[k].o * plans[k].o * 8, cudaMemcpyDeviceToHost, st));
            }
            SIE_CUDA(cudaStreamSynchronize(st));
        }
        return SIE_OK;
    } catch (const std::bad_alloc&) {
        return SIE_ENOMEM;
    }
}

int sie_dfmp2_plan_reset(sie_dfmp2_plan_t plan) {
    if (!plan) return SIE_EINVAL;
    plan->covered.clear();
    plan->covered_rows = 0;
    plan->c_ready_ws = nullptr;
    plan->dC_occ = plan->dC_vir = nullptr;
    return SIE_OK;
}

int sie_dfmp2_destroy(sie_dfmp2_plan_t plan) {
    if (!plan) return SIE_OK;
    if (plan->copy_stream) {
        cudaStreamSynchronize(plan->copy_stream);
        for (int i = 0; i < 2; ++i) {
            cudaEventDestroy(plan->ev_ready[i]);
            cudaEventDestroy(plan->ev_consumed[i]);
        }
        cudaEventDestroy(plan->ev_fork);
        for (cudaEvent_t e : plan->ev_chunk) cudaEventDestroy(e);
        cudaStreamDestroy(plan->copy_stream);
    }
    delete plan;
    return SIE_OK;
}

const char* sie_dfmp2_strerror(int status) {
    switch (status) {
        case SIE_OK: return "success";
        case SIE_EINVAL: return "invalid argument";
        case SIE_ENOMEM: return "out of memory or workspace too small";
        case SIE_ECUDA: return "CUDA error";
        case SIE_ESTATE: return "invalid call order";
        case SIE_EGAP: return "orbital gap violated: max(e_occ) >= min(e_vir)";
        case SIE_EUNSUPPORTED: return "no compute-capability-10.x CUDA device";
        case SIE_ETOOBIG: return "problem exceeds the static scratch of the no-allocation entry point";
        default: return "unknown status";
    }
}

const char* sie_dfmp2_last_cuda_error(void) { return g_last_error.c_str(); }

unsigned long long sie_dfmp2_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

static int timing_out(Prof& prof, double* ms, int n) {
    double t[ST_COUNT], c[ST_COUNT];
    SIE_TRY(prof.collect(t, c));
    for (int k = 0; k < n && k < 2 * ST_COUNT; ++k)
        if (ms) ms[k] = k < ST_COUNT ? t[k] : c[k - ST_COUNT];
    return SIE_OK;
}

int sie_dfmp2_plan_timing(sie_dfmp2_plan_t plan, double* ms, int n) {
    if (!plan || !ms || n < 0) return SIE_EINVAL;
    if (!plan->prof.on) return SIE_ESTATE;
    return timing_out(plan->prof, ms, n);
}

int sie_dfmp2_batch_timing(double* ms, int n) {
    if (!ms || n < 0) return SIE_EINVAL;
    if (!g_batch_prof.on) return SIE_ESTATE;
    return timing_out(g_batch_prof, ms, n);
}

int sie_dfmp2_probe_fp64(int kind, int iters, int ctas_per_sm, void* scratch, double* tflops, double* ms, void* cuda_stream) {
    if (!scratch || !tflops) return SIE_EINVAL;
    SIE_TRY(check_device());
    double flops = 0.0;
    float t = 0.f;
    SIE_TRY(run_probe(kind, iters, ctas_per_sm, query_num_sms(), static_cast<double*>(scratch), &flops, &t,
                      static_cast<cudaStream_t>(cuda_stream)));
    *tflops = flops / (t * 1e-3) * 1e-12;
    if (ms) *ms = t;
    return SIE_OK;
}

int sie_dfmp2_plan_info(sie_dfmp2_plan_t plan, long long* info, int n) {
    if (!plan) return 0;
    const PairGeom geo = pair_geom();
    const long long vals[8] = {plan->t8, plan->t8, plan->ta, plan->o8, (long long)plan->tiles.size(), plan->ncta, plan->pblk,
                               plan->ref ? 1 : (plan->general ? 2 : 0)};
    for (int i = 0; i < n && i < 8; ++i)
        if (info) info[i] = vals[i];
    return 8;
}

}  // extern "C"
