// noalloc.cu — sie_dfmp2_energy_noalloc: the fused pair stage + projector/trace (steps A3-A6) for callers that must not
// allocate device memory and have no workspace to hand over (code under CUDA graph capture, tight serving loops,
// harnesses that forbid cudaMalloc).  Everything the pair kernel and the reduction need beside the caller's inputs and
// outputs — the partial-G slots, the (cluster, tile) work list with its round-gate counter and the two descriptors —
// lives in ONE file-scope static device array of SIE_NOALLOC_SCRATCH_BYTES.  Every GPU that loads the library holds that
// array until the process exits.
//
// The name of a __device__ array is a host-side stand-in in host code, not a device address: the address the kernels get
// is fetched with cudaGetSymbolAddress, once per device, with that device current (scratch_base below).
//
// All calls share the array and it keeps the last call's contents: the entry point clears what must start at zero (the
// slots and the gate counter) on the caller's stream, and two calls whose work overlaps on the GPU (different streams,
// or different host threads) RACE — serialise them on one stream.
#include <algorithm>
#include <atomic>
#include <cstring>
#include <vector>

#include "../../include/sie_dfmp2.h"
#include "sie_common.cuh"
#include "sie_internal.h"

namespace sie {

static __device__ __align__(256) unsigned char g_noalloc_scratch[SIE_NOALLOC_SCRATCH_BYTES];

namespace {

// device address of g_noalloc_scratch on the CURRENT device; looked up once per device ordinal
std::atomic<unsigned char*> g_scratch_addr[64];

int scratch_base(unsigned char** out) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return set_cuda_error(e);
    const bool tracked = dev >= 0 && dev < 64;
    unsigned char* p = tracked ? g_scratch_addr[dev].load(std::memory_order_acquire) : nullptr;
    if (!p) {
        void* sym = nullptr;
        e = cudaGetSymbolAddress(&sym, g_noalloc_scratch);  // the symbol of THIS translation unit, on the current device
        if (e != cudaSuccess) return set_cuda_error(e);
        if (!sym) return set_cuda_error_text("cudaGetSymbolAddress returned a null address for the static scratch");
        p = static_cast<unsigned char*>(sym);
        if (tracked) g_scratch_addr[dev].store(p, std::memory_order_release);
    }
    *out = p;
    return SIE_OK;
}

size_t up256(size_t x) { return (x + 255) / 256 * 256; }

}  // namespace
}  // namespace sie

using namespace sie;

extern "C" {

size_t sie_dfmp2_noalloc_capacity(void) { return (size_t)SIE_NOALLOC_SCRATCH_BYTES; }

size_t sie_dfmp2_noalloc_bytes(int nocc, int nvir) {
    if (nocc < 1 || nvir < 1) return 0;
    const PairGeom geo = pair_geom();
    if (nocc > geo.TM) return 0;
    const int o8 = (nocc + 7) / 8 * 8, nst = o8 / 8;
    const int ta = std::max(1, geo.TM / nocc);
    const size_t nblk = ((size_t)nvir + ta - 1) / ta;
    const size_t ntiles = nblk * (nblk + 1) / 2;
    const int kp = nst >= geo.ncons ? 1 : geo.ncons / nst;
    const size_t slots = up256((size_t)148 * kp * o8 * o8 * 8);  // sized for the B200's 148 persistent CTAs
    return up256(sizeof(PairCluster)) + up256(sizeof(ReduceCluster)) + up256(ntiles * sizeof(PairTile) + 256) + slots;
}

int sie_dfmp2_energy_noalloc(int nocc, int nvir, int naux, const double* B, const double* e_occ, const double* e_vir,
                             const double* P_frag, double* E_out, double* G_out, void* cuda_stream) {
    if (nocc < 1 || nvir < 1 || naux < 1 || !B || !e_occ || !e_vir || !E_out) return SIE_EINVAL;
    const PairGeom geo = pair_geom();
    if (nocc > geo.TM) return SIE_EUNSUPPORTED;  // the fused kernel keeps an o x o block in one tile
    if ((reinterpret_cast<uintptr_t>(B) & 15) != 0) return SIE_EINVAL;  // TMA needs a 16-byte aligned base
    int dev = 0, sms = 0, major = 0;
    cudaError_t ce = cudaGetDevice(&dev);
    if (ce == cudaSuccess) ce = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (ce == cudaSuccess) ce = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
    if (ce != cudaSuccess) return set_cuda_error(ce);
    if (major != 10) return SIE_EUNSUPPORTED;

    // ---- the plan of sie_dfmp2_plan for the fused route, restated (host arithmetic only)
    const int o = nocc, v = nvir;
    const int o8 = (o + 7) / 8 * 8, nst = o8 / 8, naux_ld = (naux + 7) / 8 * 8;
    const int ta = std::max(1, geo.TM / o), t8 = (ta * o + 7) / 8 * 8;
    const int nblk = (v + ta - 1) / ta;
    if (nblk > 65535) return SIE_EINVAL;
    const size_t ntiles = (size_t)nblk * (nblk + 1) / 2;
    const int ncta = (int)std::min<size_t>((size_t)sms, ntiles);
    const int kp = nst >= geo.ncons ? 1 : geo.ncons / nst;
    const size_t slot_bytes = (size_t)ncta * kp * o8 * o8 * 8;

    // ---- carve the static array; refuse what does not fit
    const size_t off_desc = 0;
    const size_t off_rc = off_desc + up256(sizeof(PairCluster));
    const size_t off_tiles = off_rc + up256(sizeof(ReduceCluster));
    const size_t off_slots = off_tiles + up256(ntiles * sizeof(PairTile) + 256);  // + the round-gate counter behind the list
    const size_t need = off_slots + up256(slot_bytes);
    if (need > (size_t)SIE_NOALLOC_SCRATCH_BYTES) return SIE_ETOOBIG;
    unsigned char* base = nullptr;
    int rc = scratch_base(&base);
    if (rc != SIE_OK) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);

    // ---- descriptors and the static work list (the same enumeration as the workspace path: column groups of 12 blocks)
    PairCluster pc;
    std::memset(&pc, 0, sizeof pc);
    const uint64_t rows = (uint64_t)o * v;  // B[a][i][P] read as a plain (v*o) x naux matrix, row = a*o + i
    rc = make_tensor_map_3d(&pc.map, B, (uint64_t)naux, rows, 1, (uint64_t)naux_ld * 8, rows * naux_ld * 8, 8, (uint32_t)t8, 1);
    if (rc != SIE_OK) return rc;
    double* gpart = reinterpret_cast<double*>(base + off_slots);
    pc.e_occ = e_occ;
    pc.e_vir = e_vir;
    pc.gpart = gpart;
    pc.o = o, pc.v = v, pc.o8 = o8, pc.ta = ta;
    pc.kblocks = (naux + 7) / 8;
    pc.kp = kp;
    pc.t8 = t8;
    pc.tx_bytes = 2u * 8u * (uint32_t)t8 * 8u;
    pc.gate = 1;
    pc.mode = 0;
    std::vector<PairTile> tiles;  // host memory only
    try {
        tiles.reserve(ntiles);
    } catch (const std::bad_alloc&) {
        return SIE_ENOMEM;
    }
    const int S = 12;
    for (int J0 = 0; J0 < nblk; J0 += S) {
        const int J1 = std::min(nblk, J0 + S);
        for (int bi = 0; bi < J1; ++bi)
            for (int bj = std::max(bi, J0); bj < J1; ++bj) tiles.push_back(PairTile{0, (unsigned short)bi, (unsigned short)bj});
    }
    ReduceCluster rd{};
    rd.gpart = gpart;
    rd.P = P_frag;
    rd.E_out = E_out;
    rd.G_out = G_out;
    rd.o = o, rd.o8 = o8, rd.nslots = ncta * kp, rd.mode = 0;

    // ---- enqueue: descriptors as kernel parameters, the list by a stream-ordered copy, then clear what must start at zero
    rc = launch_poke(&pc, sizeof pc, base + off_desc, st);
    if (rc == SIE_OK) rc = launch_poke(&rd, sizeof rd, base + off_rc, st);
    if (rc != SIE_OK) return rc;
    ce = cudaMemcpyAsync(base + off_tiles, tiles.data(), tiles.size() * sizeof(PairTile), cudaMemcpyHostToDevice, st);
    if (ce == cudaSuccess) ce = cudaMemsetAsync(base + off_tiles + tiles.size() * sizeof(PairTile), 0, 256, st);
    if (ce == cudaSuccess) ce = cudaMemsetAsync(gpart, 0, slot_bytes, st);
    if (ce != cudaSuccess) return set_cuda_error(ce);
    rc = launch_pair(reinterpret_cast<const PairCluster*>(base + off_desc), reinterpret_cast<const PairTile*>(base + off_tiles), (int)ntiles,
                     ncta, t8, pair_small_strip(o, pair_producer_warp(t8) != 0) ? 3 : 0, pair_producer_warp(t8), st);
    if (rc != SIE_OK) return rc;
    return launch_reduce(reinterpret_cast<const ReduceCluster*>(base + off_rc), 1, st);
}

}  // extern "C"
