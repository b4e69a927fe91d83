// Internal declarations of libsfft_b200 (not part of the C ABI; see include/sfft.h).
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>
#include <string>
#include <vector>

#include "../../include/sfft.h"

namespace sfft {

constexpr int kProfMarks = 10;   // event marks per profiled step (see sfft_plan_profile_read)
constexpr int kMaxTile = 4;     // sequences per side of a correlation job tile
constexpr int kColsPerCta = 8;  // spectrum columns (m) per CTA in the correlation kernel

// One column-sequence fed to the x-direction correlation:  value(x, m) = xw[x] * img[x][m]
//   img >= 0 : row-transformed image `img` of the spectrum stack (0..nKy-1: g_j(y) R, nKy: S)
//   img <  0 : the constant-in-m real sequence xw[x] (a background x-basis function)
//   xw  <  0 : no x-weight (1)
struct Seq { int img; int xw; };

// A tile of (A x B) sequence pairs correlated at lags |rho| <= hw; output entries
// out_off + (ai*nb + bi)*(2hw+1) + (rho+hw)
struct Job { int na, nb, hw, out_off; int a[kMaxTile]; int b[kMaxTile]; };

// One (G entry row -> lag table row) reduction over the spectrum columns m:
//   dst[e] = (1/W) sum_m w_m Re[ G[g_entry][m] * ghat[gj][m] * exp(+2 pi i m eps / W) ],  eps = e - hw
// (ghat factor skipped when gj < 0).
struct Unit { int g_entry; int gj; int hw; int dst_off; };

struct DeviceTables {
    double *xwt = nullptr;      // [nKa + nBa][H]   x-axis basis tables (kernel rows first)
    double *gK = nullptr;       // [nKa][W]         kernel y-axis basis
    double *gB = nullptr;       // [nBa][W]         background y-axis basis
    double2 *twW = nullptr;     // [W]              exp(-2 pi i k / W)
    double2 *ghatB = nullptr;   // [nBa][W/2+1]     DFT_y of gB rows (half spectrum)
    double *phi0 = nullptr;     // [FB][FB]         M_bb (plan constant)
    Seq *seqs = nullptr;
    Job *jobs = nullptr;
    Unit *units = nullptr;
    int *kti = nullptr, *ktj = nullptr, *bti = nullptr, *btj = nullptr;
};

}  // namespace sfft

struct sfft_plan {
    int H = 0, W = 0, L = 0, w = 0, DK = 0, DB = 0, basis = 0, nbatch = 1;
    int FK = 0, FB = 0, nKa = 0, nBa = 0, n = 0, Nh = 0;
    int nimg = 0;        // spectrum stack depth per batch entry: nKa weighted-y images + S
    int gcols = 0;       // padded column count of G rows (>= W/2+1)
    int nentries = 0;    // G rows per batch entry
    int npairs = 0;      // FK(FK+1)/2
    int ldl = 0;         // leading dimension of the Cholesky factor buffer (>= n+1)
    int LT = 0;          // padded tap width of the subtract kernel instantiation (>= L)
    std::vector<int> kti, ktj, bti, btj;
    std::vector<sfft::Seq> seqs;
    std::vector<sfft::Job> jobs;
    std::vector<sfft::Unit> units;
    sfft::DeviceTables dt;
    // lag-table layout (doubles per batch entry)
    size_t off_om = 0, off_th = 0, off_la = 0, off_de = 0, tab_size = 0;
    // workspace partition (device pointers into the caller's buffer)
    void *ws = nullptr; size_t ws_bytes = 0;
    double2 *rhat = nullptr; double2 *G = nullptr; double *tab = nullptr;
    double *M = nullptr, *rhs = nullptr, *Lf = nullptr, *dscale = nullptr, *kfold = nullptr, *ctab = nullptr;
    double *stageR = nullptr, *stageS = nullptr, *stageD = nullptr, *stageC = nullptr;
    int *flag = nullptr;
    cudaStream_t stream = nullptr;
    bool built = false, solved = false;
    long launches = 0;
    int prof_steps = 0, prof_cur = -1;          // stage profiling (sfft_plan_profile)
    std::vector<cudaEvent_t> prof_events;       // [prof_steps][kProfMarks]
    std::string cuda_err;
};

namespace sfft {
// stage launchers (each returns cudaError_t of the launch); all enqueue on p->stream
cudaError_t launch_rowfft_forward(sfft_plan *p, const double *dR, const double *dS);
cudaError_t launch_corr(sfft_plan *p);
cudaError_t launch_lagsum(sfft_plan *p);
cudaError_t launch_gather(sfft_plan *p);
cudaError_t launch_solve(sfft_plan *p, double *d_coef);
int subtract_tap_width(int L);
void prof_mark(sfft_plan *p, int mark);
cudaError_t launch_subtract(sfft_plan *p, const double *d_coef, const double *dR, const double *dS, double *dD);
}  // namespace sfft
