// Steps a3+a4: cross-spectra and the "saccadic" restriction to the kernel lags.
//
// After the row transform (rowfft.cu) every correlation array of App. B
// factorises over the spectrum columns m:
//   Omega_{tb,t}(rho,eps) = sum_{x,y} R^tb(x,y) R^t(x+rho,y+eps)                              (B6, DESIGN g2)
//     = (1/W) sum_m w_m Re[ G_{tb,t}(rho; m) exp(+2 pi i m eps / W) ],   w_0 = w_{W/2} = 1, else 2
//   G_{tb,t}(rho; m) = sum_x conj(A_tb(x,m)) B_t((x+rho) mod H, m),     A_t(x,m) = f_i(x) r_j(x,m)
// and likewise Theta (B = S, B14), Lambda (B = background function, whose row transform is the
// rank-1 product f'_i(x) ghat'_j(m), B8) and Delta (B16).  Only |rho| <= L-1 (Omega) or <= w
// (the others) is ever read by the normal matrix (B5-B15), so the x-direction is evaluated at
// those lags only and the full-size correlation arrays of the paper are never materialised.
//
// k_corr_lags : G[b][entry][m]  (this file's hot kernel; FP64-FMA bound)
// k_lagsum    : the m-sum above -> lag tables Omega / Theta / Lambda / Delta
#include "sfft_internal.h"

namespace sfft {
namespace {

constexpr int XT = 32;   // rows of x per shared-memory tile

// value of sequence `sq` at (x, column m): xw[x] * img[x][m] with the packed DC/Nyquist slot undone
__device__ __forceinline__ double2 load_seq(const double2 *__restrict__ rhat_b, const double *__restrict__ xwt, Seq sq,
                                            int x, int m, int H, int Nh) {
    double wgt = sq.xw >= 0 ? __ldg(&xwt[(size_t)sq.xw * H + x]) : 1.0;
    if (sq.img < 0) return make_double2(wgt, 0.0);
    if (m > Nh) return make_double2(0.0, 0.0);
    const double2 *col = rhat_b + ((size_t)sq.img * H + x) * Nh;
    double2 v;
    if (m == 0) v = make_double2(__ldg(&col[0]).x, 0.0);
    else if (m == Nh) v = make_double2(__ldg(&col[0]).y, 0.0);
    else v = __ldg(&col[m]);
    return make_double2(v.x * wgt, v.y * wgt);
}

// grid: x = column chunk (kColsPerCta columns), y = job, z = batch.  block: (kColsPerCta, 2*hwmax+1)
__global__ void k_corr_lags(const double2 *__restrict__ rhat, const double *__restrict__ xwt,
                            const Seq *__restrict__ seqs, const Job *__restrict__ jobs, double2 *__restrict__ G,
                            int H, int Nh, int nimg, int nentries, int gcols, int hwmax) {
    extern __shared__ double2 sm[];
    const Job job = jobs[blockIdx.y];
    const int c = threadIdx.x, ri = threadIdx.y, MC = kColsPerCta;
    const int m0 = blockIdx.x * MC, hw = job.hw, nlag = 2 * hw + 1;
    const int brows = XT + 2 * hwmax;
    double2 *As = sm;                          // [kMaxTile][XT][MC]
    double2 *Bs = sm + kMaxTile * XT * MC;     // [kMaxTile][brows][MC]
    const double2 *rhat_b = rhat + (size_t)blockIdx.z * nimg * H * Nh;
    const int tid = threadIdx.y * MC + threadIdx.x, nthr = blockDim.x * blockDim.y;

    double2 acc[kMaxTile][kMaxTile];
#pragma unroll
    for (int i = 0; i < kMaxTile; ++i)
#pragma unroll
        for (int j = 0; j < kMaxTile; ++j) acc[i][j] = make_double2(0.0, 0.0);

    for (int x0 = 0; x0 < H; x0 += XT) {
        __syncthreads();
        for (int i = tid; i < job.na * XT * MC; i += nthr) {
            int cc = i % MC, r = (i / MC) % XT, s = i / (MC * XT);
            As[(s * XT + r) * MC + cc] = load_seq(rhat_b, xwt, seqs[job.a[s]], x0 + r, m0 + cc, H, Nh);
        }
        const int nbr = XT + 2 * hw;
        for (int i = tid; i < job.nb * nbr * MC; i += nthr) {
            int cc = i % MC, r = (i / MC) % nbr, s = i / (MC * nbr);
            int x = (x0 + r - hw) & (H - 1);
            Bs[(s * brows + r) * MC + cc] = load_seq(rhat_b, xwt, seqs[job.b[s]], x, m0 + cc, H, Nh);
        }
        __syncthreads();
        if (ri < nlag) {
#pragma unroll 4
            for (int r = 0; r < XT; ++r) {
                double2 a[kMaxTile], b[kMaxTile];
#pragma unroll
                for (int i = 0; i < kMaxTile; ++i) a[i] = As[(i * XT + r) * MC + c];
#pragma unroll
                for (int j = 0; j < kMaxTile; ++j) b[j] = Bs[(j * brows + r + ri) * MC + c];
#pragma unroll
                for (int i = 0; i < kMaxTile; ++i)
#pragma unroll
                    for (int j = 0; j < kMaxTile; ++j) {   // acc += conj(a) * b
                        acc[i][j].x = fma(a[i].x, b[j].x, fma(a[i].y, b[j].y, acc[i][j].x));
                        acc[i][j].y = fma(a[i].x, b[j].y, fma(-a[i].y, b[j].x, acc[i][j].y));
                    }
            }
        }
    }
    if (ri < nlag && m0 + c <= Nh) {
        double2 *Gb = G + (size_t)blockIdx.z * nentries * gcols;
#pragma unroll
        for (int i = 0; i < kMaxTile; ++i)
#pragma unroll
            for (int j = 0; j < kMaxTile; ++j)
                if (i < job.na && j < job.nb)
                    Gb[(size_t)(job.out_off + (i * job.nb + j) * nlag + ri) * gcols + m0 + c] = acc[i][j];
    }
}

// One CTA per (unit, batch): dst[e] = (1/W) sum_m w_m Re[G[m] ghat[m] exp(+2 pi i m (e-hw)/W)]
__global__ void k_lagsum(const double2 *__restrict__ G, const Unit *__restrict__ units,
                         const double2 *__restrict__ ghatB, const double2 *__restrict__ twW, double *__restrict__ tab,
                         int Nh, int W, int nentries, int gcols, size_t tab_size) {
    extern __shared__ double2 row[];   // [Nh+1]
    const Unit u = units[blockIdx.x];
    const double2 *g = G + ((size_t)blockIdx.y * nentries + u.g_entry) * gcols;
    const int Wh1 = Nh + 1;
    const double inv = 1.0 / (double)W;
    for (int m = threadIdx.x; m < Wh1; m += blockDim.x) {
        double2 v = g[m];
        if (u.gj >= 0) {
            double2 h = __ldg(&ghatB[(size_t)u.gj * Wh1 + m]);
            v = make_double2(v.x * h.x - v.y * h.y, v.x * h.y + v.y * h.x);
        }
        double wm = (m == 0 || m == Nh) ? inv : 2.0 * inv;
        row[m] = make_double2(v.x * wm, v.y * wm);
    }
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
    const int neps = 2 * u.hw + 1;
    double *dst = tab + (size_t)blockIdx.y * tab_size + u.dst_off;
    for (int e = warp; e < neps; e += nwarp) {
        const int eps = e - u.hw;
        double s = 0.0;
        for (int m = lane; m < Wh1; m += 32) {
            // exp(+2 pi i m eps / W) = conj(twW[(m*eps) mod W])
            double2 t = __ldg(&twW[(m * eps) & (W - 1)]);
            double2 v = row[m];
            s += v.x * t.x + v.y * t.y;     // Re[v * conj(t)]
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
        if (lane == 0) dst[e] = s;
    }
}

}  // namespace

cudaError_t launch_corr(sfft_plan *p) {
    const int hwmax = p->L - 1, MC = kColsPerCta;
    size_t smem = (size_t)(kMaxTile * XT * MC + kMaxTile * (XT + 2 * hwmax) * MC) * sizeof(double2);
    cudaError_t e = cudaFuncSetAttribute(k_corr_lags, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    dim3 grid((p->Nh + 1 + MC - 1) / MC, (unsigned)p->jobs.size(), p->nbatch), block(MC, 2 * hwmax + 1);
    k_corr_lags<<<grid, block, smem, p->stream>>>(p->rhat, p->dt.xwt, p->dt.seqs, p->dt.jobs, p->G, p->H, p->Nh,
                                                  p->nimg, p->nentries, p->gcols, hwmax);
    p->launches++;
    return cudaGetLastError();
}

cudaError_t launch_lagsum(sfft_plan *p) {
    size_t smem = (size_t)(p->Nh + 1) * sizeof(double2);
    cudaError_t e = cudaFuncSetAttribute(k_lagsum, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    dim3 grid((unsigned)p->units.size(), p->nbatch);
    k_lagsum<<<grid, 128, smem, p->stream>>>(p->G, p->dt.units, p->dt.ghatB, p->dt.twW, p->tab, p->Nh, p->W,
                                             p->nentries, p->gcols, p->tab_size);
    p->launches++;
    return cudaGetLastError();
}

}  // namespace sfft
