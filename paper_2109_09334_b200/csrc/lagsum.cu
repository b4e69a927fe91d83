// Step a4 (y-direction): the pruned inverse DFT over the spectrum columns m.  Each lag-table row is
//   dst[eps + hw] = (1/W) sum_m w_m Re[ G[e][m] exp(+2 pi i m (sgn eps) / W) ],  |eps| <= hw      (B6, B14)
// with G the per-column lag sums of corr.cu (summed here over the Sx partial x-ranges).  Because
// cos is even and sin odd in eps, one pass over G yields
//   P[k] = sum_m Re G[m] c(m,k),  Q[k] = sum_m Im G[m] s(m,k),  k = 0..L-1,   (c,s) = w_m (cos,sin)(2 pi m k/W)/W
// and every output is  P[|eps|] - sign(sgn eps) Q[|eps|]:  only 2L-1 of the W inverse-DFT outputs
// are ever formed ("saccadic" along y).
//
// k_lagsum_partial : thread = G entry e (coalesced along e), CTA = a chunk of kLagChunk columns;
//                    writes part[b][chunk][k][P|Q][e]
// k_lagsum_final   : thread = one lag-table value; adds the chunk partials in a fixed order
//                    (deterministic) and applies the sign rule.
#include "sfft_internal.h"

namespace sfft {
namespace {

template <int LP>
__global__ void __launch_bounds__(128) k_lagsum_partial(const double2 *__restrict__ G, const double2 *__restrict__ lagtw,
                                                        double *__restrict__ part, int Nh, int L, int E, int Sx, int nch,
                                                        int chunk) {
    __shared__ double2 tw[kLagChunk][LP];
    const int e = blockIdx.x * 128 + threadIdx.x, ch = blockIdx.y, bz = blockIdx.z;
    const int mbeg = ch * chunk, mcnt = min(chunk, Nh + 1 - mbeg);      // chunk <= kLagChunk, a multiple of 8
    for (int i = threadIdx.x; i < chunk * LP; i += 128) {
        const int mm = i / LP, k = i % LP;
        tw[mm][k] = (mm < mcnt && k < L) ? __ldg(&lagtw[(size_t)(mbeg + mm) * L + k]) : make_double2(0.0, 0.0);
    }
    __syncthreads();
    if (e >= E) return;
    double P[LP], Q[LP];
#pragma unroll
    for (int k = 0; k < LP; ++k) P[k] = Q[k] = 0.0;
    for (int xs = 0; xs < Sx; ++xs) {
        const double2 *g = G + (((size_t)bz * Sx + xs) * (Nh + 1) + mbeg) * E + e;
        // eight column loads in flight per thread (the loop is otherwise one L2 round trip per column)
        for (int m8 = 0; m8 < mcnt; m8 += 8) {
            double2 v[8];
#pragma unroll
            for (int q = 0; q < 8; ++q) v[q] = (m8 + q < mcnt) ? g[(size_t)(m8 + q) * E] : make_double2(0.0, 0.0);
#pragma unroll
            for (int q = 0; q < 8; ++q) {
#pragma unroll
                for (int k = 0; k < LP; ++k) {
                    const double2 t = tw[m8 + q][k];
                    P[k] = fma(v[q].x, t.x, P[k]);
                    Q[k] = fma(v[q].y, t.y, Q[k]);
                }
            }
        }
    }
    double *dst = part + (((size_t)bz * nch + ch) * L) * 2 * E + e;
#pragma unroll
    for (int k = 0; k < LP; ++k)
        if (k < L) { dst[(size_t)(2 * k) * E] = P[k]; dst[(size_t)(2 * k + 1) * E] = Q[k]; }
}

template <int NF>
__global__ void k_lagsum_final(const double *__restrict__ part, const LagUnit *__restrict__ units, double *__restrict__ tab,
                               int nunits, int nO, int L, int E, int nch, size_t tab_size) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x, bz = blockIdx.y;
    if (i >= nunits * nO) return;
    const LagUnit u = units[i / nO];
    const int j = i % nO;
    if (j > 2 * u.hw) return;
    const int eps = j - u.hw, k = eps < 0 ? -eps : eps;
    const double *src = part + ((size_t)bz * nch * L + k) * 2 * E + u.e;
    double P = 0.0, Q = 0.0;
    // NF partials (2 NF loads) in flight per thread.  Many chunks and few outputs (single large frames): NF = 32, the
    // kernel is a handful of L2 round trips long; few chunks and many outputs (batches of small frames): NF = 8, the
    // kernel is throughput bound and lives on occupancy.  Same summation order either way (deterministic).
    for (int c8 = 0; c8 < nch; c8 += NF) {
        double p8[NF], q8[NF];
#pragma unroll
        for (int q = 0; q < NF; ++q) {
            const bool ok = c8 + q < nch;
            p8[q] = ok ? src[(size_t)(c8 + q) * L * 2 * E] : 0.0;
            q8[q] = ok ? src[(size_t)(c8 + q) * L * 2 * E + E] : 0.0;
        }
#pragma unroll
        for (int q = 0; q < NF; ++q) { P += p8[q]; Q += q8[q]; }
    }
    const int s = (eps == 0) ? 0 : ((eps > 0) == (u.sgn > 0) ? 1 : -1);
    tab[(size_t)bz * tab_size + u.dst_off + j] = P - s * Q;
}

template <int LP>
cudaError_t launch_partial(sfft_plan *p) {
    dim3 grid((p->E + 127) / 128, p->nch, p->nbatch);
    k_lagsum_partial<LP><<<grid, 128, 0, p->stream>>>(p->G, p->dt.lagtw, p->lagpart, p->Nh, p->L, p->E, p->Sx, p->nch,
                                                     p->lagchunk);
    p->launches++;
    return cudaGetLastError();
}

}  // namespace

cudaError_t launch_lagsum(sfft_plan *p) {
    cudaError_t e;
    if (p->L <= 1) e = launch_partial<1>(p);
    else if (p->L <= 9) e = launch_partial<9>(p);
    else if (p->L <= 17) e = launch_partial<17>(p);
    else if (p->L <= 25) e = launch_partial<25>(p);
    else e = launch_partial<33>(p);
    if (e != cudaSuccess) return e;
    const int nO = 2 * p->L - 1, total = (int)p->units.size() * nO;
    dim3 grid((total + 255) / 256, p->nbatch);
    if (p->nch > 32)
        k_lagsum_final<32><<<grid, 256, 0, p->stream>>>(p->lagpart, p->dt.units, p->tab, (int)p->units.size(), nO, p->L, p->E,
                                                       p->nch, p->tab_size);
    else
        k_lagsum_final<8><<<grid, 256, 0, p->stream>>>(p->lagpart, p->dt.units, p->tab, (int)p->units.size(), nO, p->L, p->E,
                                                      p->nch, p->tab_size);
    p->launches++;
    return cudaGetLastError();
}

}  // namespace sfft
