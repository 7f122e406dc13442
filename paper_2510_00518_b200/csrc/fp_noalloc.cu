// fp_noalloc.cu -- fp_kappa_rta_static: the RTA conductivity (a9 of SURVEY.md §8(a)) for callers that
// cannot allocate -- code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
//
// fp_kappa_rta sums all modes in one CTA and, for host buffers, stages them in the context's workspace scratch.  The
// variant here is a multi-CTA reduction whose scratch -- the staged rates (host buffers only), the per-CTA partial
// sums, the device-side result and a ticket counter -- lives in ONE file-scope device array of a fixed size (below),
// which every GPU that loads the library holds until the process exits.  The entry point calls no cudaMalloc /
// cudaFree and no allocating library routine.
//
// Every call shares the array: calls that overlap on the GPU (two streams, two host threads, two contexts on one
// device) race on it.  It keeps the last call's contents; the only word that must start at zero, the ticket counter,
// is cleared by a memset node at the start of every call (and reset by the kernel's last CTA).
#include <mutex>

#include "fp_device.cuh"

namespace {

constexpr int NA_MAXM = FP_NOALLOC_MAX_MODES;  // largest N*nb the entry point accepts
constexpr int NA_BLOCKS = 64, NA_T = 256;      // CTAs x threads of the reduction
// layout of the scratch, in doubles: [0, NA_MAXM) staged Gamma_total | 16: kappa (9 used) | NA_BLOCKS*9 partial sums |
// 2: ticket counter (an unsigned in the first word)
constexpr size_t NA_OFF_KAPPA = NA_MAXM, NA_OFF_PART = NA_OFF_KAPPA + 16, NA_OFF_TICKET = NA_OFF_PART + NA_BLOCKS * 9;
constexpr size_t NA_DOUBLES = NA_OFF_TICKET + 2;

static __device__ __align__(256) double g_noalloc_scratch[NA_DOUBLES];   // 529,040 bytes per device

// In host code the array's name is a host-side stand-in, not a device address: the address is looked up once per device,
// with that device current, and cached.
std::mutex g_na_mu;
double *g_na_addr[64] = {};

cudaError_t noalloc_scratch(int dev, double **out) {
    std::lock_guard<std::mutex> lock(g_na_mu);
    if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
    if (!g_na_addr[dev]) {
        void *p = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&p, g_noalloc_scratch);   // (the caller has checked that `dev` is current)
        if (e != cudaSuccess) return e;
        g_na_addr[dev] = static_cast<double *>(p);
    }
    *out = g_na_addr[dev];
    return cudaSuccess;
}

// kappa^{ab} = pref sum_lambda f(f+1) omega^2 v^a v^b / Gamma_lambda, zero modes and modes with Gamma <= 0 skipped
// (k_kappa, fp_kernels.cu), as a two-level sum in a fixed order: grid-stride slices -> fixed-order block sums -> the
// last CTA to finish (ticket) adds the partial sums in CTA order.  Deterministic run to run.
__global__ void __launch_bounds__(NA_T) k_kappa_static(FpDev d, const double *gamma_total, double pref, double *part,
                                                        unsigned *ticket, double *kappa) {
    __shared__ double sh[32];
    __shared__ bool last;
    double acc[9];
    for (int x = 0; x < 9; x++) acc[x] = 0.0;
    const int nmodes = d.N * d.nb;
    for (int m = blockIdx.x * blockDim.x + threadIdx.x; m < nmodes; m += gridDim.x * blockDim.x) {
        const ModeRec r = d.rec[m];
        const double g = gamma_total[m];
        if (r.omega == 0.0 || !(g > 0.0)) continue;
        const double fo = d.occ[m];
        const double c = fo * (fo + 1.0) * r.omega * r.omega / g;
        const double v[3] = {r.vx, r.vy, r.vz};
        for (int a = 0; a < 3; a++)
            for (int b = 0; b < 3; b++) acc[3 * a + b] = fma(c * v[a], v[b], acc[3 * a + b]);
    }
    for (int x = 0; x < 9; x++) {
        const double tot = block_sum<double>(acc[x], sh);
        if (threadIdx.x == 0) part[blockIdx.x * 9 + x] = tot;
    }
    if (threadIdx.x == 0) {
        __threadfence();                                              // the partial sums are visible before the ticket
        last = atomicAdd(ticket, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!last) return;
    __threadfence();
    if (threadIdx.x < 9) {
        const volatile double *p = part;
        double s = 0.0;
        for (unsigned b = 0; b < gridDim.x; b++) s += p[b * 9 + threadIdx.x];
        kappa[threadIdx.x] = pref * s;
    }
    if (threadIdx.x == 0) *ticket = 0u;                               // ready for the next call
}

}  // namespace

extern "C" int fp_kappa_rta_static(fp_ctx *ctx, const double *gamma_total, double *kappa, fp_memloc loc, void *stream) {
    if (!ctx) return FP_EINVAL;
    auto fail = [&](int code, const std::string &msg) { ctx->err = msg; return code; };
    if (!gamma_total || !kappa) return fail(FP_EINVAL, "null argument");
    const FpDev &d = ctx->d;
    const size_t M = (size_t)d.N * d.nb;
    if (M > (size_t)NA_MAXM)
        return fail(FP_EINVAL, "fp_kappa_rta_static: " + std::to_string(M) + " modes exceed the static scratch of FP_NOALLOC_MAX_MODES = " +
                                   std::to_string(NA_MAXM) + " modes (use fp_kappa_rta)");
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(FP_ECUDA, std::string("cudaGetDevice: ") + cudaGetErrorString(e));
    if (dev != ctx->device) return fail(FP_ESTATE, "the context was set up on device " + std::to_string(ctx->device) + ", which is not current");
    double *scr = nullptr;
    e = noalloc_scratch(dev, &scr);
    if (e != cudaSuccess) return fail(FP_ECUDA, std::string("cudaGetSymbolAddress: ") + cudaGetErrorString(e));
#define NA_CU(call)                                                                                      \
    do {                                                                                                 \
        cudaError_t e_ = (call);                                                                         \
        if (e_ != cudaSuccess) return fail(FP_ECUDA, std::string(#call) + ": " + cudaGetErrorString(e_)); \
    } while (0)
    cudaStream_t st = (cudaStream_t)stream;
    double cst[4];
    fp_constants(cst);                                                // [2] = C_kappa
    const double pref = cst[2] / (d.T * d.T * ctx->vol * (double)d.N);
    unsigned *ticket = reinterpret_cast<unsigned *>(scr + NA_OFF_TICKET);
    NA_CU(cudaMemsetAsync(ticket, 0, sizeof(unsigned), st));          // the one word that must start at zero
    const double *g = gamma_total;
    double *k = kappa;
    if (loc == FP_MEM_HOST) {
        NA_CU(cudaMemcpyAsync(scr, gamma_total, M * sizeof(double), cudaMemcpyHostToDevice, st));
        g = scr; k = scr + NA_OFF_KAPPA;
    }
    k_kappa_static<<<NA_BLOCKS, NA_T, 0, st>>>(d, g, pref, scr + NA_OFF_PART, ticket, k);
    NA_CU(cudaGetLastError());
    if (loc == FP_MEM_HOST) {
        NA_CU(cudaMemcpyAsync(kappa, k, 9 * sizeof(double), cudaMemcpyDeviceToHost, st));
        NA_CU(cudaStreamSynchronize(st));
    }
#undef NA_CU
    return FP_OK;
}
