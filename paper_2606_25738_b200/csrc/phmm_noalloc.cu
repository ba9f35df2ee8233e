// phmm_forward_batch_noalloc: the PHMM_FP64 computation of short-class pairs through an entry point that allocates NOTHING
// (no cudaMalloc / cudaFree / allocating library routine, no context): for callers under CUDA graph capture, tight serving
// loops, harnesses that forbid allocation.  Declared in include/pairhmm_b200.h.
//
// The kernel is a variant of the fp64 sub-warp kernel k_rescue_f64t<double> (phmm_rescue.cu; SURVEY.md section 8(a) rows
// a3-a5, a9: the T/J engine in double on a row-constant table in double) without the device-side binning: one warp = one
// pair, its ceil(k / 32) first lanes active.  What that kernel keeps in workspaces of the context -- the 10^(-q/10)
// tables and the row-constant table, 64 bytes per read row -- lives here in ONE file-scope array of PHMM_NOALLOC_SCRATCH_BYTES
// (8 MiB; every GPU that loads the library holds it until exit).  Its name is a host-side stand-in in host code, not a device
// address: the address is taken once per device with cudaGetSymbolAddress (noalloc_setup) and passed to the kernels.
//
// Every call shares the array, which keeps the last call's contents: the zero run of the table (what lanes outside their
// stream read) is cleared on every call, every entry a kernel reads is rewritten before it is read (stream order).  Two calls
// that overlap on the GPU (different streams, no dependency) RACE on it: serialise them.
#include <math.h>
#include <string.h>

#include <mutex>

#include "../../include/pairhmm_b200.h"
#include "phmm_batcher.h"
#include "phmm_common.cuh"
#include "phmm_kernels.h"

namespace phmm {

constexpr size_t NOALLOC_LUT_BYTES = 4096;  // 512 doubles: [0..255] gap qualities, [256..511] base qualities
constexpr int64_t NOALLOC_MAX_ENTRIES = (PHMM_NOALLOC_SCRATCH_BYTES - NOALLOC_LUT_BYTES) / 64;

static __device__ __align__(256) unsigned char g_noalloc_scratch[PHMM_NOALLOC_SCRATCH_BYTES];

struct RawD { double gam, A, C, G, pm, px; uint32_t w; };

// One warp per pair (grid-stride over the pairs).  flags[pair] = 0, or PHMM_FLAG_RANGE where the unscaled double (scale
// constant 2^1000, reading G2) could not represent the likelihood (the value written is then -inf or inaccurate).
__global__ void __launch_bounds__(128, 2) k_noalloc_f64(DevBatch b, const double* __restrict__ table, const int* __restrict__ pair_read,
                                                         const int* __restrict__ pair_hap, int n_pairs, double* __restrict__ out,
                                                         uint8_t* __restrict__ flags) {
    constexpr int NV = RESCUE_NV;
    constexpr int LOG2C = 1000;
    const int lane = threadIdx.x & 31;
    const int warps = gridDim.x * (blockDim.x >> 5);
    const double LOG10_2 = 0.30102999566398119521;
    for (int pair = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); pair < n_pairs; pair += warps) {
        const int r = pair_read[pair], h = pair_hap[pair];
        const int64_t ro = b.read_off[r], ho = b.hap_off[h];
        const int l = (int)(b.read_off[r + 1] - ro), k = (int)(b.hap_off[h + 1] - ho);
        const int run0 = (int)(table_run_start(ro, r) - b.table_base);
        const int g = (k + NV - 1) / NV;  // lanes that hold columns (k <= 32 * NV: checked by the entry point)
        const bool active = lane < g;
        const int n_ent = l + 2;          // run-in entry, rows 1..l, sum entry
        const int steps = n_ent + g - 1;  // lane L runs one entry behind lane L-1

        // haplotype columns of this lane: one match word per base code, [4] = N; [5] = what "matches" the sum entry
        // (prior pm = 0): the columns more than one behind the haplotype's last (phmm_engine.cuh)
        const int j0 = lane * NV;
        const int nv = active ? min(max(k - j0, 0), NV) : 0;
        uint32_t hm[6] = {0u, 0u, 0u, 0u, 0u, 0u};
        for (int x = 0; x < nv; x++) {
            const int c = base_code(b.hap_bases[ho + j0 + x]);
#pragma unroll
            for (int q = 0; q < 5; q++) hm[q] |= (c == q ? 1u : 0u) << x;
        }
#pragma unroll
        for (int x = 0; x < NV; x++) hm[5] |= (j0 + x > k ? 1u : 0u) << x;
        const bool is_last = lane == g - 1;
        const bool full_last = k == g * NV;
        const double Cok = ldexp(1.0, LOG2C) / (double)k;  // Eq.1 with C = 2^1000

        double T[NV], J[NV];
#pragma unroll
        for (int x = 0; x < NV; x++) { T[x] = 0.0; J[x] = 0.0; }
        double outS = 0.0, outT = 0.0;

        // entry e of the pair's run (e < 0 or e >= n_ent: an all-zero entry of the table's zero run); layout: k_table_f64
        auto fetch = [&](RawD& re, int e) {
            const int pos = (active && (unsigned)e < (unsigned)n_ent) ? run0 + e : 0;
            const double* q = table + (((int64_t)(pos >> 5)) << 8) + (pos & 31);
            re.gam = __ldg(q); re.A = __ldg(q + 32); re.C = __ldg(q + 64); re.G = __ldg(q + 96);
            re.pm = __ldg(q + 128); re.px = __ldg(q + 160);
            re.w = __ldg(reinterpret_cast<const uint32_t*>(q - (pos & 31) + 192) + (pos & 31));
        };
        RawD cur, nxt;
        fetch(cur, -lane);
        for (int s = 0; s < steps; s++) {
            fetch(nxt, s + 1 - lane);
            const double gam = cur.gam, A = cur.A, C = cur.C, G = cur.G, pm = cur.pm, px = cur.px;
            const uint32_t meta = cur.w & 0xffu;
            const uint32_t code = meta & META_CODE_MASK;
            const uint32_t m01 = (code & 1u) ? hm[1] : hm[0], m23 = (code & 1u) ? hm[3] : hm[2];
            uint32_t mw = (code & 4u) ? hm[4] : ((code & 2u) ? m23 : m01);  // Eq.3, literal: N matches N only
            mw = (meta & META_SUM) ? hm[5] : mw;
            const double prevT = outT;
            double inS = __shfl_up_sync(PHMM_FULL, outS, 1), inT = __shfl_up_sync(PHMM_FULL, prevT, 1);
            if (lane == 0) {  // column-0 boundary, Eq.1 (reading G1): only the run-in entry injects
                inS = (meta & META_FIRST) ? Cok : 0.0;
                inT = C * inS;
            }
            double sr = inS;
            double U = ((mw & 1u) ? pm : px) * T[0];
            T[0] = inT;
#pragma unroll
            for (int x = 0; x < NV; x++) {  // the T/J step of phmm_engine.cuh: 4 FMA + 1 MUL per cell
                double Un = U;
                if (x + 1 < NV) Un = ((mw & (1u << (x + 1))) ? pm : px) * T[x + 1];
                const double Wv = fma(A, U, J[x]);
                const double Tn = fma(C, sr, Wv);
                J[x] = fma(G, J[x], U);
                sr = fma(gam, sr, U);
                if (x + 1 < NV) T[x + 1] = Tn; else outT = Tn;
                U = Un;
            }
            outS = sr;
            if (is_last && (meta & META_SUM)) {  // Eq.4: the running sum has collected M_l + I_l of every column
                const double sig = full_last ? outS + prevT : outS;
                out[pair] = log10(sig) - (double)LOG2C * LOG10_2;
                if (flags) flags[pair] = (sig >= 1e-290 && sig < 1e300) ? 0 : PHMM_FLAG_RANGE;
            }
            cur = nxt;
        }
        __syncwarp();
    }
}

// ---- set-up, once per device: the array's device address, the quality tables
namespace {
struct NoallocDev { unsigned char* base = nullptr; int n_sm = 0; bool ready = false; };
NoallocDev g_dev[64];
std::mutex g_mu;

struct DevGuard {  // makes `device` current for the call, restores the caller's device afterwards
    int prev = -1;
    bool ok = false;
    explicit DevGuard(int device) {
        if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
        ok = (prev == device) || cudaSetDevice(device) == cudaSuccess;
        if (prev == device) prev = -1;
    }
    ~DevGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

int noalloc_setup(int device) {  // with `device` current
    if (device < 0 || device >= 64) return PHMM_E_ARG;
    std::lock_guard<std::mutex> lock(g_mu);
    NoallocDev& d = g_dev[device];
    if (d.ready) return PHMM_OK;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return PHMM_E_CUDA;
    if (prop.major != 10) return PHMM_E_UNSUPPORTED;
    void* ptr = nullptr;
    if (cudaGetSymbolAddress(&ptr, g_noalloc_scratch) != cudaSuccess || !ptr) return PHMM_E_CUDA;
    // 10^(-q/10), the paper's "q64" table: raw Phred bytes, no floor (the defaults of phmm_options)
    double lut[512];
    for (int q = 0; q < 256; q++) lut[q] = lut[256 + q] = pow(10.0, -(double)q / 10.0);
    if (cudaMemcpy(ptr, lut, sizeof(lut), cudaMemcpyHostToDevice) != cudaSuccess) return PHMM_E_CUDA;
    d.base = (unsigned char*)ptr;
    d.n_sm = prop.multiProcessorCount;
    d.ready = true;
    return PHMM_OK;
}
}  // namespace

}  // namespace phmm

using namespace phmm;

extern "C" int phmm_noalloc_setup(int device) {
    DevGuard guard(device);
    if (!guard.ok) return PHMM_E_CUDA;
    return noalloc_setup(device);
}

extern "C" int phmm_noalloc_limits(int64_t* max_table_entries, int32_t* max_hap_len, int32_t* max_read_len) {
    if (max_table_entries) *max_table_entries = NOALLOC_MAX_ENTRIES;
    if (max_hap_len) *max_hap_len = RESCUE_MAX_K;
    if (max_read_len) *max_read_len = RESCUE_MAX_L;
    return PHMM_OK;
}

extern "C" int phmm_forward_batch_noalloc(int device, const phmm_batch* b, const int64_t* d_read_off, const int64_t* d_hap_off,
                                          const int32_t* d_pair_read, const int32_t* d_pair_hap, double* d_out_log10,
                                          uint8_t* d_out_flags, void* cuda_stream) {
    if (!b || b->n_pairs < 0 || b->n_reads < 0 || b->n_haps < 0) return PHMM_E_ARG;
    if (b->n_pairs == 0) return PHMM_OK;
    if (!d_out_log10 || !d_read_off || !d_hap_off || !d_pair_read || !d_pair_hap || !b->d_read_bases || !b->d_qual_base ||
        !b->d_qual_ins || !b->d_qual_del || !b->d_qual_gcp || !b->d_hap_bases)
        return PHMM_E_ARG;
    HostBatchView hv = {b->n_reads, b->n_haps, b->n_pairs, b->h_read_off, b->h_hap_off, b->h_pair_read, b->h_pair_hap};
    int rc = validate_batch(hv);
    if (rc != PHMM_OK) return rc;
    // ---- sizes against the fixed capacity: nothing is launched for a batch that does not fit
    int max_l = 0;  // (the table is built for every read of the batch, the limits apply to the pairs)
    for (int64_t r = 0; r < b->n_reads; r++) max_l = (int)std::max<int64_t>(max_l, b->h_read_off[r + 1] - b->h_read_off[r]);
    for (int64_t p = 0; p < b->n_pairs; p++) {
        const int r = b->h_pair_read[p], h = b->h_pair_hap[p];
        if (b->h_read_off[r + 1] - b->h_read_off[r] > RESCUE_MAX_L) return PHMM_E_TOOLONG;  // read longer than 4096
        if (b->h_hap_off[h + 1] - b->h_hap_off[h] > RESCUE_MAX_K) return PHMM_E_TOOLONG;   // haplotype longer than 1024
    }
    const int64_t table_base = table_run_start(b->h_read_off[0], 0) - TABLE_ZERO_RUN;
    const int64_t n_entries = table_run_start(b->h_read_off[b->n_reads], b->n_reads) - table_base + 2;
    if (n_entries > NOALLOC_MAX_ENTRIES) return PHMM_E_TOOLONG;  // sum of (read length + 4) beyond the scratch array
    DevGuard guard(device);
    if (!guard.ok) return PHMM_E_CUDA;
    rc = noalloc_setup(device);
    if (rc != PHMM_OK) return rc;
    const NoallocDev& d = g_dev[device];
    const double* lut = reinterpret_cast<const double*>(d.base);
    double* table = reinterpret_cast<double*>(d.base + NOALLOC_LUT_BYTES);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    DevBatch db;
    memset(&db, 0, sizeof(db));
    db.read_bases = b->d_read_bases; db.qual_base = b->d_qual_base; db.qual_ins = b->d_qual_ins;
    db.qual_del = b->d_qual_del; db.qual_gcp = b->d_qual_gcp; db.hap_bases = b->d_hap_bases;
    db.read_off = d_read_off; db.hap_off = d_hap_off;
    db.n_reads = b->n_reads; db.n_haps = b->n_haps;
    db.n_wild = 0;
    db.table_base = table_base;
    // the zero run is cleared (inside launch_table_f64), every run is rewritten: nothing of the previous call is read
    if (launch_table_f64(db, lut, table, 0, b->n_reads, max_l, st) != cudaSuccess) return PHMM_E_CUDA;
    const int64_t want = (b->n_pairs + 3) / 4;
    const int grid = (int)(want < (int64_t)d.n_sm * 8 ? want : (int64_t)d.n_sm * 8);
    k_noalloc_f64<<<grid, 128, 0, st>>>(db, table, d_pair_read, d_pair_hap, (int)b->n_pairs, d_out_log10, d_out_flags);
    return cudaGetLastError() == cudaSuccess ? PHMM_OK : PHMM_E_CUDA;
}
