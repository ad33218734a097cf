// frost_noalloc.cu -- frost_acc_noalloc: the Newtonian all-pairs sweep (Eq. 24) for
// callers that are not allowed to allocate device memory.
//
// Who that is: code that runs where a cudaMalloc / cudaFree is forbidden or unaffordable -- inside a
// region of an application whose memory is managed by a pool that owns the whole device (an allocation
// behind the pool's back can fail or fragment it), inside a latency-critical loop where the implicit
// device-wide synchronisation of cudaFree is unacceptable, or in a host program that is handed a fixed
// memory budget up front.  Everything else in this library goes through a frost_ctx whose scratch
// buffers grow on demand with cudaMalloc (frost_common.cuh: ensure()); this file is the one entry point
// that never does.
//
// How: it is a variant of the one-sided Newton sweep (frost_sweeps.cu: sweep_kernel<NewtonPolicy> +
// reduce_vec_kernel).  That sweep needs scratch beyond its inputs and outputs -- the packed source
// records and one partial sum per (source slice, sink) -- and here the scratch is the file-scope
// __device__ array g_scratch below: a fixed sizeof(g_scratch) = 6.5 MiB that every GPU on which this
// library's module is loaded holds until the process exits.  The price is the size limit
// FROST_NOALLOC_MAX_N.
//
// Rules that follow from one shared static array (also stated in include/frost.h):
//   * All calls on one device use the same array, and it keeps whatever the previous call left in it.
//     Nothing in it needs to start at zero: each call rewrites every record it will read (padding
//     records included) and every partial sum it will add, before reading them, on its own stream.
//   * Two calls that overlap on the GPU (different streams, or different host threads without
//     ordering between their streams) race on the array.  Serialise them.
//   * In host code the name g_scratch is a host-side shadow symbol, not a device address: a kernel
//     that received &g_scratch[0] would fault (or, on systems where the GPU can reach host memory,
//     silently use the wrong memory).  The device address is looked up once per device with
//     cudaGetSymbolAddress while that device is current, and that pointer is what the kernels get.
//   * This lookup happens in the first call on each device; it may load the module.  Make that first
//     call outside any stream capture.
#include <mutex>

#include "frost_pairs.cuh"

namespace frost {
namespace {

constexpr int kMaxN = FROST_NOALLOC_MAX_N;            // 16384 particles
constexpr int kMaxSlices = 16;                        // source slices (partial sums per sink)
constexpr int kNT = 128;                              // threads per CTA, one sink each
constexpr size_t kRecDoubles = (size_t)kMaxN * 4;                 // packed {x,y,z,m}: 512 KiB
constexpr size_t kPartDoubles = (size_t)kMaxSlices * 3 * kMaxN;   // [slice][plane][sink]: 6 MiB
constexpr size_t kScratchDoubles = kRecDoubles + kPartDoubles;
constexpr int kMaxDevices = 64;

static_assert(kMaxN % kTile == 0 && kMaxN % kNT == 0, "padding of the record stream");

// The scratch.  Device code of this file could name it directly; host code must not (see above).
static __device__ __align__(256) double g_scratch[kScratchDoubles];

std::mutex g_mu;
double *g_dev_ptr[kMaxDevices] = {};   // device address of g_scratch, per device ordinal

// records k < n: {x, y, z, m} of particle k; records n .. n_pad-1: zero mass at the origin (they are
// read as sources and as sinks of the last blocks, and must not carry a previous call's particles)
__global__ void noalloc_pack_kernel(int n, int n_pad, int ld, const double *__restrict__ pos,
                                    const double *__restrict__ mass, double4 *__restrict__ rec) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_pad) return;
    rec[k] = k < n ? make_double4(pos[k], pos[(size_t)ld + k], pos[2 * (size_t)ld + k], mass[k])
                   : make_double4(0.0, 0.0, 0.0, 0.0);
}

// grid = (n_pad / kNT sink blocks, slices).  Sources arrive in shared memory by 1-D TMA bulk copies
// through a kStages ring, as in sweep_kernel; every pair goes through NewtonPolicy::pair.
__global__ void __launch_bounds__(kNT, 4) noalloc_newton_kernel(const SweepParams prm) {
    __shared__ __align__(128) double4 tiles[kStages][kTile];
    __shared__ __align__(8) uint64_t full[kStages];
    const int tid = threadIdx.x;
    const int tile0 = blockIdx.y * prm.tiles_per_slice;
    const int ntiles = min(prm.tiles_per_slice, prm.n_tiles - tile0);

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < kStages; ++s) mbar_init(&full[s], 1);
        mbar_fence_init();
    }
    __syncthreads();
    auto issue = [&](int t) {
        const int s = t % kStages;
        mbar_expect_tx(&full[s], kTile * kRecBytes);
        bulk_g2s(&tiles[s][0], prm.src0 + (size_t)(tile0 + t) * kTile, kTile * kRecBytes, &full[s]);
    };
    if (tid == 0)
        for (int t = 0; t < min(kStages - 1, ntiles); ++t) issue(t);

    NewtonPolicy::Sink snk;
    NewtonPolicy::Acc acc;
    const int i = blockIdx.x * kNT + tid;
    NewtonPolicy::load(snk, prm, i);
    NewtonPolicy::init(acc);

    for (int t = 0; t < ntiles; ++t) {
        // every thread has finished tile t-1, whose stage is the one refilled now
        __syncthreads();
        if (tid == 0 && t + kStages - 1 < ntiles) issue(t + kStages - 1);
        const int s = t % kStages;
        mbar_wait(&full[s], (uint32_t)(t / kStages) & 1u);
#pragma unroll 4
        for (int j = 0; j < kTile; ++j) {
            const double4 r = tiles[s][j];
            NewtonPolicy::pair(snk, acc, r, r, prm);
        }
    }
    NewtonPolicy::store(acc, prm.partial + (size_t)blockIdx.y * 3 * prm.n_pad, prm.n_pad, i);
}

// out_acc[c*ld + i] = G * (partials of sink i added in ascending slice order)
__global__ void noalloc_reduce_kernel(const double *__restrict__ partial, int n_pad, int slices, int n,
                                      double G, int ld, double *__restrict__ out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double sx = 0.0, sy = 0.0, sz = 0.0;
    for (int s = 0; s < slices; ++s) {
        const double *p = partial + (size_t)s * 3 * n_pad;
        sx += p[i]; sy += p[n_pad + i]; sz += p[2 * n_pad + i];
    }
    out[i] = G * sx; out[(size_t)ld + i] = G * sy; out[2 * (size_t)ld + i] = G * sz;
}

struct CurrentDevice {      // make `device` current for the call, restore the caller's on return
    int prev = -1;
    cudaError_t err = cudaSuccess;
    explicit CurrentDevice(int device) {
        err = cudaGetDevice(&prev);
        if (err == cudaSuccess && prev != device) err = cudaSetDevice(device);
        else prev = -1;
    }
    ~CurrentDevice() { if (prev >= 0) cudaSetDevice(prev); }
};

// Device address of g_scratch on `device` (which is current).  First call per device only.
cudaError_t scratch_address(int device, double **out) {
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_dev_ptr[device]) {
        double *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void **)&p, g_scratch);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_dev_ptr[device] = p;
    }
    *out = g_dev_ptr[device];
    return cudaSuccess;
}

}  // namespace
}  // namespace frost

extern "C" {

int frost_noalloc_max_n(void) { return frost::kMaxN; }

int frost_acc_noalloc(int device, void *stream, int n, int ld, const double *pos, const double *mass,
                      double G, double eps2, double *out_acc, int *cuda_error) {
    using namespace frost;
    if (cuda_error) *cuda_error = 0;
    if (n < 0 || ld < n || device < 0 || device >= kMaxDevices || !(eps2 >= 0.0)) return FROST_EINVAL;
    if (n > kMaxN) return FROST_ETOOBIG;
    if (n == 0) return FROST_OK;
    if (!pos || !mass || !out_acc) return FROST_EINVAL;

#define NOALLOC_CUDA(call)                                   \
    do {                                                     \
        const cudaError_t e_ = (call);                       \
        if (e_ != cudaSuccess) {                             \
            if (cuda_error) *cuda_error = (int)e_;           \
            return FROST_ECUDA;                              \
        }                                                    \
    } while (0)

    CurrentDevice cur(device);
    NOALLOC_CUDA(cur.err);
    double *scratch = nullptr;
    NOALLOC_CUDA(scratch_address(device, &scratch));
    cudaStream_t st = (cudaStream_t)stream;

    const int n_pad = round_up(n, kTile);                     // multiple of kTile and of kNT
    const int n_tiles = n_pad / kTile;
    const int slices = n_tiles < kMaxSlices ? n_tiles : kMaxSlices;
    double4 *rec = (double4 *)scratch;
    double *partial = scratch + kRecDoubles;

    noalloc_pack_kernel<<<(n_pad + 255) / 256, 256, 0, st>>>(n, n_pad, ld, pos, mass, rec);
    NOALLOC_CUDA(cudaGetLastError());

    SweepParams prm{};
    prm.snk0 = prm.src0 = rec;
    prm.partial = partial; prm.n_pad = n_pad;
    prm.n_tiles = n_tiles; prm.tiles_per_slice = (n_tiles + slices - 1) / slices;
    // floor as in sweep_newton: the self pair (and a coincident unsoftened one) then has a finite
    // weight and a zero separation, and adds nothing (frost.h conventions)
    prm.eps2 = eps2 > 0x1p-400 ? eps2 : 0x1p-400;
    prm.G = G;
    const int used = (n_tiles + prm.tiles_per_slice - 1) / prm.tiles_per_slice;   // non-empty slices
    noalloc_newton_kernel<<<dim3(n_pad / kNT, used), kNT, 0, st>>>(prm);
    NOALLOC_CUDA(cudaGetLastError());

    noalloc_reduce_kernel<<<(n + 255) / 256, 256, 0, st>>>(partial, n_pad, used, n, G, ld, out_acc);
    NOALLOC_CUDA(cudaGetLastError());
#undef NOALLOC_CUDA
    return FROST_OK;
}

}  // extern "C"
