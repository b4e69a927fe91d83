// NEXT-2: crowded-flavor preprocessing (reading DESIGN g21).  "The crowded-flavor SFFT will
// automatically mask the pixels affected by the saturated sources in the field and replace them with the
// neighboring background"; the fit then runs on the masked pair and the solution is applied to the original pair.
//   seed = R >= sat_R or S >= sat_S;  mask = seed grown by rd pixels (square window, wrap-around);
//   masked pixels of each image <- mean of its unmasked pixels in the (2 rb + 1)^2 window around them
//   (no unmasked pixel there: mean of all unmasked pixels of the image); unmasked pixels are copied.
// The square growth is separable (rows, then columns).  HBM-bound streaming passes over the pair; the fill gathers
// only at the (few) masked pixels.
#include <mutex>

#include "sfft_internal.h"

namespace sfft {
namespace {

// t(x,y) = OR_{|dy| <= rd} seed(x, (y+dy) mod W)
__global__ void k_mask_rows(const double *__restrict__ R, const double *__restrict__ S, unsigned char *__restrict__ t,
                            int H, int W, int rd, double satR, double satS) {
    const int y = blockIdx.x * blockDim.x + threadIdx.x, x = blockIdx.y, b = blockIdx.z;
    if (y >= W) return;
    const size_t row = ((size_t)b * H + x) * W;
    int m = 0;
    for (int dy = -rd; dy <= rd; ++dy) {
        const int yy = wrap_index(y + dy, W, (W & (W - 1)) == 0 ? W - 1 : -1);
        m |= (__ldg(&R[row + yy]) >= satR) | (__ldg(&S[row + yy]) >= satS);
    }
    t[row + y] = (unsigned char)m;
}

// mask(x,y) = OR_{|dx| <= rd} t((x+dx) mod H, y)
__global__ void k_mask_cols(const unsigned char *__restrict__ t, unsigned char *__restrict__ mask, int H, int W, int rd) {
    const int y = blockIdx.x * blockDim.x + threadIdx.x, x = blockIdx.y, b = blockIdx.z;
    if (y >= W) return;
    const size_t img = (size_t)b * H * W;
    int m = 0;
    for (int dx = -rd; dx <= rd; ++dx) m |= t[img + (size_t)(wrap_index(x + dx, H, (H & (H - 1)) == 0 ? H - 1 : -1)) * W + y];
    mask[img + (size_t)x * W + y] = (unsigned char)m;
}

// partial sums of the unmasked pixels: part[b][blk] = (sum R, sum S, count), fixed order (deterministic)
__global__ void __launch_bounds__(256) k_unmasked_partial(const double *__restrict__ R, const double *__restrict__ S,
                                                          const unsigned char *__restrict__ mask, double *__restrict__ part,
                                                          size_t P, int nblk) {
    const int b = blockIdx.y, tid = threadIdx.x;
    const size_t chunk = (P + nblk - 1) / nblk, lo = (size_t)blockIdx.x * chunk, hi = lo + chunk < P ? lo + chunk : P;
    double sr = 0.0, ss = 0.0, cnt = 0.0;
    for (size_t i = lo + tid; i < hi; i += 256) {
        const size_t q = (size_t)b * P + i;
        if (!mask[q]) { sr += R[q]; ss += S[q]; cnt += 1.0; }
    }
    __shared__ double red[3][256];
    red[0][tid] = sr; red[1][tid] = ss; red[2][tid] = cnt;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (tid < o) { red[0][tid] += red[0][tid + o]; red[1][tid] += red[1][tid + o]; red[2][tid] += red[2][tid + o]; }
        __syncthreads();
    }
    if (tid < 3) part[((size_t)b * nblk + blockIdx.x) * 3 + tid] = red[tid][0];
}

// gmean[b] = (mean R, mean S) over the unmasked pixels
__global__ void k_unmasked_mean(const double *__restrict__ part, double *__restrict__ gmean, int nblk) {
    const int b = blockIdx.x;
    if (threadIdx.x != 0) return;
    double sr = 0.0, ss = 0.0, cnt = 0.0;
    for (int k = 0; k < nblk; ++k) { sr += part[((size_t)b * nblk + k) * 3]; ss += part[((size_t)b * nblk + k) * 3 + 1]; cnt += part[((size_t)b * nblk + k) * 3 + 2]; }
    gmean[2 * b] = cnt > 0.0 ? sr / cnt : 0.0;
    gmean[2 * b + 1] = cnt > 0.0 ? ss / cnt : 0.0;
}

// copy / fill.  Rm may alias R (and Sm alias S): only unmasked pixels are read from the window and those are never modified.
__global__ void k_fill(const double *R, const double *S, const unsigned char *__restrict__ mask,
                       const double *__restrict__ gmean, double *Rm, double *Sm, int H, int W, int rb) {
    const int y = blockIdx.x * blockDim.x + threadIdx.x, x = blockIdx.y, b = blockIdx.z;
    if (y >= W) return;
    const size_t img = (size_t)b * H * W, p = img + (size_t)x * W + y;
    if (!mask[p]) {
        const double r = R[p], s = S[p];
        Rm[p] = r; Sm[p] = s;
        return;
    }
    double sr = 0.0, ss = 0.0;
    int cnt = 0;
    for (int dx = -rb; dx <= rb; ++dx) {
        const size_t row = img + (size_t)(wrap_index(x + dx, H, (H & (H - 1)) == 0 ? H - 1 : -1)) * W;
        for (int dy = -rb; dy <= rb; ++dy) {
            const size_t q = row + (wrap_index(y + dy, W, (W & (W - 1)) == 0 ? W - 1 : -1));
            if (!mask[q]) { sr += R[q]; ss += S[q]; ++cnt; }
        }
    }
    Rm[p] = cnt > 0 ? sr / cnt : gmean[2 * b];
    Sm[p] = cnt > 0 ? ss / cnt : gmean[2 * b + 1];
}

}  // namespace

cudaError_t launch_mask_fill(sfft_plan *p, const double *dR, const double *dS, double satR, double satS, int rd, int rb,
                             double *dRm, double *dSm, unsigned char *dmask) {
    const int H = p->H, W = p->W, nb = p->nbatch;
    const size_t P = (size_t)H * W;
    // scratch in the spectrum-stack region of the workspace (rewritten by the next build): row-grown seeds, partial sums
    unsigned char *t = reinterpret_cast<unsigned char *>(p->rhat);
    const int nblk = 256;
    double *part = reinterpret_cast<double *>(t + (((size_t)nb * P + 255) & ~(size_t)255));
    double *gmean = part + (size_t)nb * nblk * 3;
    dim3 grid((W + 255) / 256, H, nb);
    k_mask_rows<<<grid, 256, 0, p->stream>>>(dR, dS, t, H, W, rd, satR, satS);
    k_mask_cols<<<grid, 256, 0, p->stream>>>(t, dmask, H, W, rd);
    k_unmasked_partial<<<dim3(nblk, nb), 256, 0, p->stream>>>(dR, dS, dmask, part, P, nblk);
    k_unmasked_mean<<<nb, 32, 0, p->stream>>>(part, gmean, nblk);
    k_fill<<<grid, 256, 0, p->stream>>>(dR, dS, dmask, gmean, dRm, dSm, H, W, rb);
    p->launches += 5;
    return cudaGetLastError();
}

}  // namespace sfft

// ---- sfft_mask_fill_static: the mask/fill of one pair with its scratch inside the library image ---------------
// For callers that cannot give the library device memory and must not have it allocate any (a process whose memory
// all belongs to one pool, a loop that may not stall on cudaMalloc's device-wide synchronisation): no plan, no
// workspace, no cudaMalloc / cudaFree.  The kernels are the ones launch_mask_fill runs; only the scratch differs.
constexpr size_t kStaticHead = 8192;      // partial sums [256][3] doubles (6144 B) + the two means, rounded up
constexpr int kStaticMaxDev = 64;

// Scratch of sfft_mask_fill_static: [0, kStaticHead) partial sums and means, then one flag byte per pixel.  Shared by
// every call on the device and never cleared (each call writes what it reads).  Costs its size on every GPU that loads
// this library, until the process exits.
static __device__ __align__(256) unsigned char g_static_scratch[kStaticHead + SFFT_STATIC_MAX_PIXELS];

namespace {

// In host code `g_static_scratch` is only a handle for the runtime, not somewhere a kernel may write: the address
// kernels get is asked for once per device (with that device current) and kept here.
std::mutex g_static_mu;
unsigned char *g_static_ptr[kStaticMaxDev] = {};
thread_local std::string g_static_err;

int static_fail(int status, const std::string &msg) {
    g_static_err = msg;
    return status;
}

}  // namespace

extern "C" const char *sfft_static_last_error(void) { return g_static_err.c_str(); }

extern "C" int sfft_mask_fill_static(const double *d_R, const double *d_S, int H, int W, double sat_R, double sat_S,
                                     int rd, int rb, double *d_Rm, double *d_Sm, unsigned char *d_mask,
                                     void *cuda_stream) {
    if (!d_R || !d_S || !d_Rm || !d_Sm || !d_mask)
        return static_fail(SFFT_ERR_INVALID_ARG, "sfft_mask_fill_static: null image pointer");
    if (H < 1 || W < 1 || H > 16384 || W > 16384 || (long)H * (long)W > SFFT_STATIC_MAX_PIXELS)
        return static_fail(SFFT_ERR_INVALID_ARG,
                           "sfft_mask_fill_static: frame of " + std::to_string(H) + " x " + std::to_string(W) +
                               " pixels exceeds the built-in scratch (1 <= H, W <= 16384 and H*W <= " +
                               std::to_string(SFFT_STATIC_MAX_PIXELS) + "); use sfft_mask_fill with a workspace");
    if (rd < 0 || rd > 64 || rb < 1 || rb > 128 || !(sat_R == sat_R) || !(sat_S == sat_S))
        return static_fail(SFFT_ERR_INVALID_ARG, "sfft_mask_fill_static: need 0 <= rd <= 64, 1 <= rb <= 128, sat_* not NaN");
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return static_fail(SFFT_ERR_CUDA, std::string("cudaGetDevice: ") + cudaGetErrorString(e));
    if (dev < 0 || dev >= kStaticMaxDev) return static_fail(SFFT_ERR_CUDA, "sfft_mask_fill_static: device ordinal above 63");
    unsigned char *scratch = nullptr;
    {
        std::lock_guard<std::mutex> lock(g_static_mu);
        if (!g_static_ptr[dev]) {       // first call on this device: its copy of the array has its own address
            void *sym = nullptr;
            e = cudaGetSymbolAddress(&sym, g_static_scratch);
            if (e != cudaSuccess || !sym) {
                cudaGetLastError();
                return static_fail(SFFT_ERR_CUDA, std::string("cudaGetSymbolAddress(scratch): ") + cudaGetErrorString(e));
            }
            g_static_ptr[dev] = static_cast<unsigned char *>(sym);
        }
        scratch = g_static_ptr[dev];
    }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const int nblk = 256;
    double *part = reinterpret_cast<double *>(scratch), *gmean = part + (size_t)nblk * 3;
    unsigned char *t = scratch + kStaticHead;
    const dim3 grid((W + 255) / 256, H, 1);
    sfft::k_mask_rows<<<grid, 256, 0, st>>>(d_R, d_S, t, H, W, rd, sat_R, sat_S);
    sfft::k_mask_cols<<<grid, 256, 0, st>>>(t, d_mask, H, W, rd);
    sfft::k_unmasked_partial<<<dim3(nblk, 1), 256, 0, st>>>(d_R, d_S, d_mask, part, (size_t)H * W, nblk);
    sfft::k_unmasked_mean<<<1, 32, 0, st>>>(part, gmean, nblk);
    sfft::k_fill<<<grid, 256, 0, st>>>(d_R, d_S, d_mask, gmean, d_Rm, d_Sm, H, W, rb);
    e = cudaGetLastError();
    if (e != cudaSuccess) return static_fail(SFFT_ERR_CUDA, std::string("sfft_mask_fill_static launch: ") + cudaGetErrorString(e));
    return SFFT_OK;
}
