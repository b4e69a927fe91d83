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

constexpr int kMfBlocks = 1184;      // CTAs of the unmasked-sum kernel (8 per SM); fixed, so the sums are reproducible

// t(x,y) = OR_{|dy| <= rd} seed(x, (y+dy) mod W).  A thread owns 4 consecutive pixels of a row and slides along it,
// keeping the distance to the last seed seen: 4 + 2 rd loads per image instead of 4 (2 rd + 1).
__global__ void __launch_bounds__(256) k_mask_rows(const double *__restrict__ R, const double *__restrict__ S,
                                                   unsigned char *__restrict__ t, int H, int W, int rd, double satR, double satS) {
    const int y0 = 4 * (blockIdx.x * blockDim.x + threadIdx.x), x = blockIdx.y, b = blockIdx.z;
    if (y0 >= W) return;
    const size_t row = ((size_t)b * H + x) * W;
    const int wm = (W & (W - 1)) == 0 ? W - 1 : -1;
    int since = 1 << 20;                                  // pixels since the last seed
    for (int i = -rd; i < 4 + rd; ++i) {
        const int yy = wrap_index(y0 + i, W, wm);
        const bool seed = (__ldg(&R[row + yy]) >= satR) | (__ldg(&S[row + yy]) >= satS);
        since = seed ? 0 : since + 1;
        const int yc = y0 + i - rd;                       // its window [yc - rd, yc + rd] ends at the pixel just read
        if (i >= rd && yc < W) t[row + yc] = (unsigned char)(since <= 2 * rd);
    }
}

// mask(x,y) = OR_{|dx| <= rd} t((x+dx) mod H, y).  A thread owns two adjacent columns (one 16-bit word: W is even,
// so every row starts on an even byte) and 16 consecutive rows, sliding down: 16 + 2 rd loads for 32 pixels.
constexpr int kMfColRows = 16;
__global__ void __launch_bounds__(128) k_mask_cols(const unsigned char *__restrict__ t, unsigned char *__restrict__ mask,
                                                   int H, int W, int rd) {
    const int yp = blockIdx.x * blockDim.x + threadIdx.x, x0 = blockIdx.y * kMfColRows, b = blockIdx.z;
    if (2 * yp >= W) return;
    const int hm = (H & (H - 1)) == 0 ? H - 1 : -1, W2 = W / 2;
    const unsigned short *t2 = reinterpret_cast<const unsigned short *>(t) + (size_t)b * H * W2;
    unsigned short *m2 = reinterpret_cast<unsigned short *>(mask) + (size_t)b * H * W2;
    int since0 = 1 << 20, since1 = 1 << 20;               // rows since byte 0 / byte 1 of the pair was last set
    for (int i = -rd; i < kMfColRows + rd; ++i) {
        const int xx = x0 + i;
        const unsigned short v = t2[(size_t)wrap_index(xx, H, hm) * W2 + yp];
        since0 = (v & 0x00ff) ? 0 : since0 + 1;
        since1 = (v & 0xff00) ? 0 : since1 + 1;
        // row xc = xx - rd has its whole window [xc - rd, xc + rd] = [xx - 2 rd, xx] loaded once i >= rd
        const int xc = xx - rd;
        if (i >= rd && xc < H) {
            const unsigned short o = (unsigned short)((since0 <= 2 * rd ? 1 : 0) | (since1 <= 2 * rd ? 0x100 : 0));
            m2[(size_t)xc * W2 + yp] = o;
        }
    }
}

// partial sums of the unmasked pixels: part[b][blk] = (sum R, sum S, count), fixed order (deterministic).  Two pixels
// per thread and step (P is even), loads issued whether or not the pixel is masked so that several are in flight.
__global__ void __launch_bounds__(256) k_unmasked_partial(const double *__restrict__ R, const double *__restrict__ S,
                                                          const unsigned char *__restrict__ mask, double *__restrict__ part,
                                                          size_t P, int nblk) {
    const int b = blockIdx.y, tid = threadIdx.x;
    const size_t P2 = P / 2, chunk = (P2 + nblk - 1) / nblk, lo = (size_t)blockIdx.x * chunk, hi = lo + chunk < P2 ? lo + chunk : P2;
    const double2 *R2 = reinterpret_cast<const double2 *>(R + (size_t)b * P), *S2 = reinterpret_cast<const double2 *>(S + (size_t)b * P);
    const unsigned short *M2 = reinterpret_cast<const unsigned short *>(mask + (size_t)b * P);
    double sr = 0.0, ss = 0.0;
    int cnt = 0;
    for (size_t i = lo + tid; i < hi; i += 4 * 256) {
        double2 r[4], s[4];
        unsigned short m[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const size_t q = i + 256 * u;
            m[u] = 0x0101;
            if (q < hi) { m[u] = M2[q]; r[u] = R2[q]; s[u] = S2[q]; }
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            if (!(m[u] & 0x00ff)) { sr += r[u].x; ss += s[u].x; ++cnt; }
            if (!(m[u] & 0xff00)) { sr += r[u].y; ss += s[u].y; ++cnt; }
        }
    }
    __shared__ double red[3][256];
    red[0][tid] = sr; red[1][tid] = ss; red[2][tid] = (double)cnt;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (tid < o) { red[0][tid] += red[0][tid + o]; red[1][tid] += red[1][tid + o]; red[2][tid] += red[2][tid + o]; }
        __syncthreads();
    }
    if (tid < 3) part[((size_t)b * nblk + blockIdx.x) * 3 + tid] = red[tid][0];
}

// gmean[b] = (mean R, mean S) over the unmasked pixels: tree sum of the nblk partials by one CTA per batch entry
__global__ void __launch_bounds__(256) k_unmasked_mean(const double *__restrict__ part, double *__restrict__ gmean, int nblk) {
    const int b = blockIdx.x, tid = threadIdx.x;
    double v[3] = {0.0, 0.0, 0.0};
    for (int k = tid; k < nblk; k += 256)
        for (int c = 0; c < 3; ++c) v[c] += part[((size_t)b * nblk + k) * 3 + c];
    __shared__ double red[3][256];
    for (int c = 0; c < 3; ++c) red[c][tid] = v[c];
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (tid < o) for (int c = 0; c < 3; ++c) red[c][tid] += red[c][tid + o];
        __syncthreads();
    }
    if (tid == 0) {
        const double cnt = red[2][0];
        gmean[2 * b] = cnt > 0.0 ? red[0][0] / cnt : 0.0;
        gmean[2 * b + 1] = cnt > 0.0 ? red[1][0] / cnt : 0.0;
    }
}

// Window mean of the unmasked pixels around masked pixel (x, y), by a whole warp: lane l takes the window positions
// l, l + 32, ... (row-major in the (2 rb + 1)^2 window) and the partial sums are combined by a butterfly, which
// leaves the same value in every lane (a + b = b + a exactly).  A single thread walking the window alone is a chain
// of (2 rb + 1)^2 dependent loads: it set the run time of the whole kernel.  Falls back to the global mean.
__device__ __forceinline__ void warp_fill_one(const double *R, const double *S, const unsigned char *__restrict__ mask,
                                              const double *__restrict__ gmean, size_t img, int x, int y, int H, int W, int rb,
                                              int b, double &outR, double &outS) {
    const int lane = threadIdx.x & 31, side = 2 * rb + 1, n = side * side;
    const int hm = (H & (H - 1)) == 0 ? H - 1 : -1, wm = (W & (W - 1)) == 0 ? W - 1 : -1;
    double sr = 0.0, ss = 0.0;
    int cnt = 0;
    for (int i = lane; i < n; i += 32) {
        const int dx = i / side - rb, dy = i % side - rb;
        const size_t q = img + (size_t)wrap_index(x + dx, H, hm) * W + wrap_index(y + dy, W, wm);
        if (!mask[q]) { sr += R[q]; ss += S[q]; ++cnt; }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        sr += __shfl_xor_sync(0xffffffffu, sr, o);
        ss += __shfl_xor_sync(0xffffffffu, ss, o);
        cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
    }
    outR = cnt > 0 ? sr / cnt : gmean[2 * b];
    outS = cnt > 0 ? ss / cnt : gmean[2 * b + 1];
}

// copy / fill, two adjacent pixels per thread (W even: 16-byte aligned pairs); the masked pixels of a warp are filled
// one after the other by the whole warp.  Rm may alias R (and Sm alias S): only unmasked pixels are read from the
// window and those are never modified.
__global__ void __launch_bounds__(256) k_fill(const double *R, const double *S, const unsigned char *__restrict__ mask,
                                              const double *__restrict__ gmean, double *Rm, double *Sm, int H, int W, int rb) {
    const int y = 2 * (blockIdx.x * blockDim.x + threadIdx.x), x = blockIdx.y, b = blockIdx.z, lane = threadIdx.x & 31;
    const bool live = y < W;                               // (no early exit: the fills below need all 32 lanes)
    const size_t img = (size_t)b * H * W, p = img + (size_t)x * W + (live ? y : 0);
    unsigned m = 0;
    double2 r = make_double2(0.0, 0.0), s = r;
    if (live) {
        m = *reinterpret_cast<const unsigned short *>(&mask[p]);
        r = *reinterpret_cast<const double2 *>(&R[p]);
        s = *reinterpret_cast<const double2 *>(&S[p]);
    }
    unsigned todo = __ballot_sync(0xffffffffu, m != 0);
    while (todo) {
        const int src = __ffs(todo) - 1;
        todo &= todo - 1;
        const unsigned ms = __shfl_sync(0xffffffffu, m, src);
        const int ys = __shfl_sync(0xffffffffu, y, src);
        double fr, fs;
        if (ms & 0x00ff) {
            warp_fill_one(R, S, mask, gmean, img, x, ys, H, W, rb, b, fr, fs);
            if (lane == src) { r.x = fr; s.x = fs; }
        }
        if (ms & 0xff00) {
            warp_fill_one(R, S, mask, gmean, img, x, ys + 1, H, W, rb, b, fr, fs);
            if (lane == src) { r.y = fr; s.y = fs; }
        }
    }
    if (live) {
        *reinterpret_cast<double2 *>(&Rm[p]) = r;
        *reinterpret_cast<double2 *>(&Sm[p]) = s;
    }
}

// ---- one-pixel-per-thread forms of the three kernels above, for odd W or image pointers that are not 16-byte aligned ----
// mask(x,y) = OR_{|dx| <= rd} t((x+dx) mod H, y)
__global__ void k_mask_cols_1(const unsigned char *__restrict__ t, unsigned char *__restrict__ mask, int H, int W, int rd) {
    const int y = blockIdx.x * blockDim.x + threadIdx.x, x = blockIdx.y, b = blockIdx.z;
    if (y >= W) return;
    const size_t img = (size_t)b * H * W;
    int m = 0;
    for (int dx = -rd; dx <= rd; ++dx) m |= t[img + (size_t)(wrap_index(x + dx, H, (H & (H - 1)) == 0 ? H - 1 : -1)) * W + y];
    mask[img + (size_t)x * W + y] = (unsigned char)m;
}

// partial sums of the unmasked pixels: part[b][blk] = (sum R, sum S, count), fixed order (deterministic)
__global__ void __launch_bounds__(256) k_unmasked_partial_1(const double *__restrict__ R, const double *__restrict__ S,
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

// copy / fill.  Rm may alias R (and Sm alias S): only unmasked pixels are read from the window and those are never modified.
__global__ void k_fill_1(const double *R, const double *S, const unsigned char *__restrict__ mask,
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


// launch sequence shared by the plan path and the static-scratch entry point
inline cudaError_t mask_fill_launches(const double *dR, const double *dS, double satR, double satS, int rd, int rb, double *dRm,
                                      double *dSm, unsigned char *dmask, int H, int W, int nb, unsigned char *t, double *part,
                                      double *gmean, cudaStream_t st) {
    const uintptr_t a16 = (uintptr_t)dR | (uintptr_t)dS | (uintptr_t)dRm | (uintptr_t)dSm;
    const bool pairs = W % 2 == 0 && (a16 & 15) == 0 && ((uintptr_t)dmask & 1) == 0 && ((uintptr_t)t & 1) == 0;
    k_mask_rows<<<dim3((W + 1023) / 1024, H, nb), 256, 0, st>>>(dR, dS, t, H, W, rd, satR, satS);
    if (pairs) {
        k_mask_cols<<<dim3((W / 2 + 127) / 128, (H + kMfColRows - 1) / kMfColRows, nb), 128, 0, st>>>(t, dmask, H, W, rd);
        k_unmasked_partial<<<dim3(kMfBlocks, nb), 256, 0, st>>>(dR, dS, dmask, part, (size_t)H * W, kMfBlocks);
    } else {
        k_mask_cols_1<<<dim3((W + 255) / 256, H, nb), 256, 0, st>>>(t, dmask, H, W, rd);
        k_unmasked_partial_1<<<dim3(kMfBlocks, nb), 256, 0, st>>>(dR, dS, dmask, part, (size_t)H * W, kMfBlocks);
    }
    k_unmasked_mean<<<nb, 256, 0, st>>>(part, gmean, kMfBlocks);
    if (pairs) k_fill<<<dim3((W / 2 + 255) / 256, H, nb), 256, 0, st>>>(dR, dS, dmask, gmean, dRm, dSm, H, W, rb);
    else k_fill_1<<<dim3((W + 255) / 256, H, nb), 256, 0, st>>>(dR, dS, dmask, gmean, dRm, dSm, H, W, rb);
    return cudaGetLastError();
}

}  // namespace

cudaError_t launch_mask_fill(sfft_plan *p, const double *dR, const double *dS, double satR, double satS, int rd, int rb,
                             double *dRm, double *dSm, unsigned char *dmask) {
    const int H = p->H, W = p->W, nb = p->nbatch;
    const size_t P = (size_t)H * W;
    // scratch in the spectrum-stack region of the workspace (rewritten by the next build): row-grown seeds, partial sums
    unsigned char *t = reinterpret_cast<unsigned char *>(p->rhat);
    double *part = reinterpret_cast<double *>(t + (((size_t)nb * P + 255) & ~(size_t)255));
    double *gmean = part + (size_t)nb * kMfBlocks * 3;
    p->launches += 5;
    return mask_fill_launches(dR, dS, satR, satS, rd, rb, dRm, dSm, dmask, H, W, nb, t, part, gmean, p->stream);
}

}  // namespace sfft

// ---- sfft_mask_fill_static: the mask/fill of one pair with its scratch inside the library image ---------------
// For callers that cannot give the library device memory and must not have it allocate any (a process whose memory
// all belongs to one pool, a loop that may not stall on cudaMalloc's device-wide synchronisation): no plan, no
// workspace, no cudaMalloc / cudaFree.  The kernels are the ones launch_mask_fill runs; only the scratch differs.
constexpr size_t kStaticHead = 32768;     // partial sums [1184][3] doubles (28416 B) + the two means, rounded up
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
    double *part = reinterpret_cast<double *>(scratch), *gmean = part + (size_t)sfft::kMfBlocks * 3;
    unsigned char *t = scratch + kStaticHead;
    e = sfft::mask_fill_launches(d_R, d_S, sat_R, sat_S, rd, rb, d_Rm, d_Sm, d_mask, H, W, 1, t, part, gmean, st);
    if (e != cudaSuccess) return static_fail(SFFT_ERR_CUDA, std::string("sfft_mask_fill_static launch: ") + cudaGetErrorString(e));
    return SFFT_OK;
}
