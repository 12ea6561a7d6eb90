// NUFFT Synthesis: Gram-corrected visibilities per level and a 3-D type-3 NUFFT with regular
// domain partitioning of the baselines and the pixels (PAPER.md:129-164 Eq. 17-21; :345-423 Section 3.4, Eq. 32-36, Alg. 3).
//
//   I_l(r_j) += sum_n V_l,n exp(i <s_j, x_n>),   x_n = b_pq = (x_p - x_q) / lambda_w,   s_j = -2 pi r_j   (reading Q18)
//
// One transform = one (input cell, output cell) pair. With x = x_c + x', s = s_c + s' (cell centres):
//   I_j = exp(i <s_j, x_c>) * F(s'_j),   F(s') = sum_n [V_n exp(i <s_c, x'_n>)] exp(i <s', x'_n>),   |x'_d| <= X_d, |s'_d| <= S_d.
// Per dimension (upsampling sigma = 2, kernel width w, "exponential of semicircle" phi(z) = exp(beta (sqrt(1 - z^2) - 1))):
//   1. spread (Eq. 33): grid of nf1 >= 2 sigma X S / pi + w points, source position x' sigma S / pi grid units from the middle;
//   2. the grid values are Fourier coefficients g_m, m in [-nf1/2, nf1/2); F(s') = [sum_m g_m exp(i m theta)] / phihat(theta),
//      theta = pi s' / (sigma S) in [-pi/sigma, pi/sigma]  (Eq. 34-35: phihat = the kernel's Fourier transform, by quadrature);
//   3. the sum over m is a type-2 transform: divide g_m by phihat(2 pi m / nf2), zero-pad to nf2 >= sigma nf1, FFT (cuFFT),
//      interpolate at theta with the same kernel.
// Grids and FFTs are complex64; coordinates, phases and the kernel's transform are fp64. The host does the cell bookkeeping
// (bounding boxes, index lists); everything that touches a visibility or a pixel value runs in the kernels below.
#include "internal.h"
#include <cufft.h>
#include <algorithm>
#include <cmath>
#include <map>
#include <new>
#include <tuple>

cudaStream_t bb_ctx_user_stream(bb_ctx* ctx);
int bb_ctx_device(bb_ctx* ctx);
void bb_ctx_ref(bb_ctx* ctx, int delta);

namespace {

constexpr int kMaxW = 12;               // kernel width (grid points) at most
constexpr int kQuad = 32;               // Gauss-Legendre nodes on [0, 1] for the kernel's Fourier transform
constexpr double kSigma = 2.0;          // upsampling of both stages
constexpr double kMaxGridBytes = 32e9;     // fine grids of all levels of one transform (complex64)

__constant__ double c_gl_x[kQuad], c_gl_w[kQuad];

struct KernelPar { int w; double beta; };

__host__ __device__ inline double es_kernel(double z, double beta) {      // z = 2 t / w in [-1, 1]
  const double a = 1.0 - z * z;
  return a > 0.0 ? exp(beta * (sqrt(a) - 1.0)) : 0.0;
}
// phihat(k) = int_{-w/2}^{w/2} phi(2 t / w) exp(i k t) dt = w int_0^1 phi(z) cos(k w z / 2) dz      (k: radians per grid point)
__device__ inline double es_hat_dev(double k, KernelPar kp) {
  double acc = 0.0;
  for (int q = 0; q < kQuad; ++q) acc += c_gl_w[q] * es_kernel(c_gl_x[q], kp.beta) * cos(0.5 * k * kp.w * c_gl_x[q]);
  return acc * kp.w;
}

// Alg. 3 l.8 / Eq. 17, 21: V'_l[p, q] = sum_k D[l, k] B[p, k] conj(B[q, k]); out [l][p + n_ant q] complex64 (fp64 sums)
__global__ void vis_kernel(const bb_c32* __restrict__ B, int ldb, const float* __restrict__ D, int ldd, int n_ant, int n_eig,
                           int n_levels, float2* __restrict__ V) {
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (int64_t)n_ant * n_ant) return;
  const int p = (int)(t % n_ant), q = (int)(t / n_ant);
  for (int l = 0; l < n_levels; ++l) {
    double re = 0.0, im = 0.0;
    for (int k = 0; k < n_eig; ++k) {
      const double d = D[l + (size_t)k * ldd];
      if (d == 0.0) continue;
      const bb_c32 a = B[p + (size_t)k * ldb], b = B[q + (size_t)k * ldb];
      re += d * ((double)a.re * b.re + (double)a.im * b.im);
      im += d * ((double)a.im * b.re - (double)a.re * b.im);
    }
    V[(size_t)l * n_ant * n_ant + t] = make_float2((float)re, (float)im);
  }
}

struct CellGeom {                       // one (input cell, output cell) pair
  double xc[3], sc[3];                  // centres of the sources (wavelengths) and of the targets' s = -2 pi r
  double pos_scale[3];                  // grid units per unit of x': sigma S_d / pi
  double theta_scale[3];                // theta per unit of s': pi / (sigma S_d)
  int nf1[3], nf2[3];
};

// Eq. 33: spread the cell's sources onto the nf1 grid, all levels: one warp per source, the w^3 taps spread over the lanes.
// idx: baseline ids (p + n_ant q) of the cell.
// Source id = collect * n_ant^2 + p + n_ant q; xyz: [collect][3][n_ant] (rotated frame), inv_wl: [collect], V: [collect][level][n_ant^2].
__global__ void spread_kernel(const int* __restrict__ idx, int n_src, const double* __restrict__ xyz, int n_ant,
                              const double* __restrict__ inv_wl, const float2* __restrict__ V, int n_levels, CellGeom g, KernelPar kp,
                              float2* __restrict__ grid) {
  __shared__ float ker_s[4][3][kMaxW];
  const int wib = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int t = blockIdx.x * 4 + wib;
  if (t >= n_src) return;                                                 // whole warps leave together
  const int n_base = n_ant * n_ant;
  const int id = idx[t], col = id / n_base, bq = id - col * n_base, p = bq % n_ant, q = bq / n_ant;
  const double* xc = xyz + (size_t)col * 3 * n_ant;
  const double iw = inv_wl[col];
  int i0[3];
  double ph = 0.0;
  for (int d = 0; d < 3; ++d) {
    const double xp = (xc[p + (size_t)d * n_ant] - xc[q + (size_t)d * n_ant]) * iw - g.xc[d];
    ph += g.sc[d] * xp;
    const double pos = xp * g.pos_scale[d] + 0.5 * g.nf1[d];              // grid units, well inside [w/2, nf1 - w/2]
    i0[d] = (int)ceil(pos - 0.5 * kp.w);
    if (lane < kp.w) ker_s[wib][d][lane] = (float)es_kernel(2.0 * (i0[d] + lane - pos) / kp.w, kp.beta);
  }
  __syncwarp();
  ph *= 0.15915494309189535;                                              // turns
  ph -= rint(ph);
  double sn, cs;
  sincospi(2.0 * ph, &sn, &cs);
  const size_t n1 = (size_t)g.nf1[0] * g.nf1[1] * g.nf1[2];
  const int w = kp.w, w3 = w * w * w;
  for (int l = 0; l < n_levels; ++l) {
    const float2 v = V[((size_t)col * n_levels + l) * n_base + bq];
    const float cr = (float)(v.x * cs - v.y * sn), ci = (float)(v.x * sn + v.y * cs);      // V exp(i <s_c, x'>)
    if (cr == 0.f && ci == 0.f) continue;
    float2* gl = grid + (size_t)l * n1;
    for (int tap = lane; tap < w3; tap += 32) {
      const int a = tap % w, b = (tap / w) % w, c = tap / (w * w);
      const float k3 = ker_s[wib][0][a] * ker_s[wib][1][b] * ker_s[wib][2][c];
      float2* dst = gl + ((size_t)(i0[2] + c) * g.nf1[1] + (i0[1] + b)) * g.nf1[0] + i0[0] + a;
      atomicAdd(&dst->x, cr * k3);
      atomicAdd(&dst->y, ci * k3);
    }
  }
}

// type-2 step 1: fine[k] = g_m / (phihat2_x[mx] phihat2_y[my] phihat2_z[mz]) at k = m mod nf2 (FFT order); fine was zeroed.
// dec_d: per-dimension arrays 1 / phihat(2 pi m / nf2_d), m = -nf1_d/2 .. nf1_d/2 - 1.
__global__ void deconv_pad_kernel(const float2* __restrict__ grid, int n_levels, CellGeom g, const double* __restrict__ dec0,
                                  const double* __restrict__ dec1, const double* __restrict__ dec2, float2* __restrict__ fine) {
  const int64_t n1 = (int64_t)g.nf1[0] * g.nf1[1] * g.nf1[2];
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n1) return;
  const int ix = (int)(t % g.nf1[0]), iy = (int)((t / g.nf1[0]) % g.nf1[1]), iz = (int)(t / ((int64_t)g.nf1[0] * g.nf1[1]));
  const double f = dec0[ix] * dec1[iy] * dec2[iz];
  const int kx = (ix - g.nf1[0] / 2 + g.nf2[0]) % g.nf2[0], ky = (iy - g.nf1[1] / 2 + g.nf2[1]) % g.nf2[1],
            kz = (iz - g.nf1[2] / 2 + g.nf2[2]) % g.nf2[2];
  const int64_t n2 = (int64_t)g.nf2[0] * g.nf2[1] * g.nf2[2];
  const int64_t o = ((int64_t)kz * g.nf2[1] + ky) * g.nf2[0] + kx;
  for (int l = 0; l < n_levels; ++l) {
    const float2 v = grid[(size_t)l * n1 + t];
    fine[(size_t)l * n2 + o] = make_float2((float)(v.x * f), (float)(v.y * f));
  }
}

// Eq. 34-35: interpolate the FFT output at theta_j, divide by the spreading kernel's transform, apply the post-phase and
// accumulate the real part into the level images: one warp per pixel — lane q evaluates quadrature node q of the kernel's
// transform (kQuad = 32) and the w^3 taps are spread over the lanes. idx: pixel ids of the output cell.
__global__ void interp_kernel(const int* __restrict__ idx, int n_tgt, const double* __restrict__ pix, int64_t ld_pix,
                              const float2* __restrict__ fine, int n_levels, CellGeom g, KernelPar kp, float* __restrict__ img,
                              int64_t img_stride) {
  static_assert(kQuad == 32, "one quadrature node per lane");
  __shared__ float ker_s[4][3][kMaxW];
  const int wib = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int t = blockIdx.x * 4 + wib;
  if (t >= n_tgt) return;
  const int j = idx[t];
  double corr = 1.0, post = 0.0;
  int i0[3];
  for (int d = 0; d < 3; ++d) {
    const double s = -6.283185307179586 * pix[j + (size_t)d * ld_pix];
    post += s * g.xc[d];
    const double theta = (s - g.sc[d]) * g.theta_scale[d];
    double hq = c_gl_w[lane] * es_kernel(c_gl_x[lane], kp.beta) * cos(0.5 * theta * kp.w * c_gl_x[lane]);
    for (int o = 16; o > 0; o >>= 1) hq += __shfl_xor_sync(0xffffffffu, hq, o);
    corr *= hq * kp.w;                                                    // phihat(theta_d)
    const double pos = theta * g.nf2[d] * 0.15915494309189535;            // fine-grid units, may be negative: periodic
    i0[d] = (int)ceil(pos - 0.5 * kp.w);
    if (lane < kp.w) ker_s[wib][d][lane] = (float)es_kernel(2.0 * (i0[d] + lane - pos) / kp.w, kp.beta);
  }
  __syncwarp();
  post *= 0.15915494309189535;
  post -= rint(post);
  double sn, cs;
  sincospi(2.0 * post, &sn, &cs);
  const int64_t n2 = (int64_t)g.nf2[0] * g.nf2[1] * g.nf2[2];
  const int w = kp.w, w3 = w * w * w;
  for (int l = 0; l < n_levels; ++l) {
    const float2* fl = fine + (size_t)l * n2;
    float re = 0.f, im = 0.f;
    for (int tap = lane; tap < w3; tap += 32) {
      const int a = tap % w, b = (tap / w) % w, c = tap / (w * w);
      const int kx = ((i0[0] + a) % g.nf2[0] + g.nf2[0]) % g.nf2[0], ky = ((i0[1] + b) % g.nf2[1] + g.nf2[1]) % g.nf2[1],
                kz = ((i0[2] + c) % g.nf2[2] + g.nf2[2]) % g.nf2[2];
      const float2 v = fl[((int64_t)kz * g.nf2[1] + ky) * g.nf2[0] + kx];
      const float k3 = ker_s[wib][0][a] * ker_s[wib][1][b] * ker_s[wib][2][c];
      re += k3 * v.x;
      im += k3 * v.y;
    }
    for (int o = 16; o > 0; o >>= 1) { re += __shfl_xor_sync(0xffffffffu, re, o); im += __shfl_xor_sync(0xffffffffu, im, o); }
    if (lane == 0) img[(size_t)l * img_stride + j] += (float)(((double)re * cs - (double)im * sn) / corr);   // Re[e^{i<s_j,x_c>} F / phihat]
  }
}

}  // namespace

// ---------------------------------------------------------------------------- host side
struct bb_nufft {
  bb_ctx* ctx = nullptr;
  int64_t n_pix = 0, pix_stride = 0;
  int n_levels = 0, n_part_in = 1, n_part_out = 1;
  KernelPar kp{};
  double* pix_dev = nullptr;            // [3][n_pix]
  float* img = nullptr;                 // [level][pix_stride]
  std::vector<double> pix_host;         // [3][n_pix], in the rotated frame
  double R[9] = {1, 0, 0, 0, 1, 0, 0, 0, 1};   // rows = the frame (e_u, e_v, e_w): e_w = mean pixel direction. <b, r> is invariant under
                                        // the rotation, and in this frame the pixels are thin along w (1 - cos(FoV / 2)), so
                                        // the unpartitioned third axis of an (n, n, 1) partition costs few grid points
  // output cells (fixed per handle): pixel ids grouped by cell, bounding boxes
  std::vector<int> out_start;           // n_cells + 1
  int* out_idx_dev = nullptr;
  std::vector<double> out_lo, out_hi;   // [cell][3]
  // per-collect scratch (grown on demand)
  float2 *V = nullptr, *grid = nullptr, *fine = nullptr;
  size_t V_cap = 0, grid_cap = 0, fine_cap = 0;
  int* in_idx_dev = nullptr; size_t in_idx_cap = 0;
  std::map<std::pair<int, int>, double*> dec;   // (nf1, nf2) -> device array of 1 / phihat(2 pi m / nf2), built once
  bb_c32* B_dev = nullptr; float* D_dev = nullptr; double* xyz_dev = nullptr;
  size_t B_cap = 0, D_cap = 0, xyz_cap = 0;
  // staged collects: their visibilities wait in V ([collect][level][n_ant^2]) until bb_nufft_get (or the source cap) runs ONE set
  // of transforms over the baselines of all of them — the paper's use of the NUFFT over all time steps
  int pend = 0, pend_n_ant = 0;
  std::vector<double> xyz_all, inv_wl_all;      // host: rotated antenna positions [collect][3][n_ant], 1 / wavelength
  double* xyz_all_dev = nullptr; double* inv_wl_dev = nullptr;
  size_t xyz_all_cap = 0, inv_wl_cap = 0;
  // cuFFT plans per fine-grid shape. They own NO work area (auto-allocation off): all of them run in fft_work, which
  // is sized before a flush launches anything and counted in the memory limit. Both caches are emptied after a flush
  // that left them above kMaxCachedPlans / kMaxCachedDec entries.
  struct FftPlan { cufftHandle handle; size_t work_bytes; };
  std::map<std::tuple<int, int, int>, FftPlan> plans;
  unsigned char* fft_work = nullptr; size_t fft_work_cap = 0;
  // bb_nufft_collect (Alg. 3 from S): eigenvalues, B = W V and level weights of the current collect, device resident
  double* lam_full = nullptr; bb_c32* B_full = nullptr; float* D_full = nullptr;
  size_t lam_full_cap = 0, B_full_cap = 0, D_full_cap = 0;
  int64_t n_transforms = 0, max_grid = 0;
};

namespace {

int next_smooth_even(int n) {           // smallest even 2^a 3^b 5^c >= n
  if (n < 2) n = 2;
  for (int m = n + (n & 1);; m += 2) {
    int r = m;
    while (r % 2 == 0) r /= 2;
    while (r % 3 == 0) r /= 3;
    while (r % 5 == 0) r /= 5;
    if (r == 1) return m;
  }
}

void gauss_legendre_01(double* x, double* w) {          // kQuad nodes and weights on [0, 1]
  const int n = kQuad;
  for (int i = 0; i < n; ++i) {
    double z = cos(3.141592653589793 * (i + 0.75) / (n + 0.5)), pp = 1.0;
    for (int it = 0; it < 100; ++it) {
      double p1 = 1.0, p2 = 0.0;
      for (int j = 0; j < n; ++j) { const double p3 = p2; p2 = p1; p1 = ((2.0 * j + 1.0) * z * p2 - j * p3) / (j + 1.0); }
      pp = n * (z * p1 - p2) / (z * z - 1.0);
      const double dz = p1 / pp;
      z -= dz;
      if (fabs(dz) < 1e-15) break;
    }
    x[i] = 0.5 * (z + 1.0);
    w[i] = 1.0 / ((1.0 - z * z) * pp * pp);              // (2 / ((1 - z^2) pp^2)) / 2: mapped to [0, 1]
  }
}

double es_hat_host(double k, KernelPar kp, const double* x, const double* w) {
  double acc = 0.0;
  for (int q = 0; q < kQuad; ++q) acc += w[q] * es_kernel(x[q], kp.beta) * cos(0.5 * k * kp.w * x[q]);
  return acc * kp.w;
}

template <class T>
int grow(T** p, size_t* cap, size_t need) {
  if (need <= *cap) return BB_OK;
  cudaFree(*p);
  *p = nullptr; *cap = 0;
  if (cudaMalloc(p, need * sizeof(T)) != cudaSuccess) { cudaGetLastError(); return BB_EALLOC; }
  *cap = need;
  return BB_OK;
}

// Regular partition of n points (coordinates c[d][i], d = 0..2) into parts x parts x 1 cells along the two widest axes:
// cell id per point, then ids grouped by cell (counting sort) with each non-empty cell's bounding box.
void partition(const double* c, int64_t n, int64_t ld, int parts, std::vector<int>& start, std::vector<int>& order,
               std::vector<double>& lo, std::vector<double>& hi) {
  double mn[3], mx[3];
  for (int d = 0; d < 3; ++d) {
    mn[d] = 1e300; mx[d] = -1e300;
    for (int64_t i = 0; i < n; ++i) { mn[d] = std::min(mn[d], c[d * ld + i]); mx[d] = std::max(mx[d], c[d * ld + i]); }
  }
  int ax[3] = {0, 1, 2};
  std::sort(ax, ax + 3, [&](int a, int b) { return mx[a] - mn[a] > mx[b] - mn[b]; });
  const int n_cells = parts * parts;
  std::vector<int> cell(n);
  start.assign(n_cells + 1, 0);
  for (int64_t i = 0; i < n; ++i) {
    int id[2];
    for (int u = 0; u < 2; ++u) {
      const int d = ax[u];
      const double ext = mx[d] - mn[d];
      int k = ext > 0 ? (int)((c[d * ld + i] - mn[d]) / ext * parts) : 0;
      id[u] = std::min(std::max(k, 0), parts - 1);
    }
    cell[i] = id[0] + parts * id[1];
    start[cell[i] + 1] += 1;
  }
  for (int k = 0; k < n_cells; ++k) start[k + 1] += start[k];
  order.resize(n);
  std::vector<int> fill(start.begin(), start.end() - 1);
  lo.assign((size_t)n_cells * 3, 1e300); hi.assign((size_t)n_cells * 3, -1e300);
  for (int64_t i = 0; i < n; ++i) {
    const int k = cell[i];
    order[fill[k]++] = (int)i;
    for (int d = 0; d < 3; ++d) { lo[k * 3 + d] = std::min(lo[k * 3 + d], c[d * ld + i]); hi[k * 3 + d] = std::max(hi[k * 3 + d], c[d * ld + i]); }
  }
}

// Frame (e_u, e_v, e_w) with e_w = the mean pixel direction (rows of R); the pixels ([3][n]) are rotated in place.
void rotate_to_mean_direction(std::vector<double>& pix, int64_t n_pix, double R[9]) {
  double m[3] = {0, 0, 0};
  for (int d = 0; d < 3; ++d) { for (int64_t i = 0; i < n_pix; ++i) m[d] += pix[(size_t)d * n_pix + i]; }
  const double nm = sqrt(m[0] * m[0] + m[1] * m[1] + m[2] * m[2]);
  if (nm > 1e-12 * (double)n_pix) {
    for (int d = 0; d < 3; ++d) R[6 + d] = m[d] / nm;
    int k = 0;                                                      // the coordinate axis least aligned with e_w
    for (int d = 1; d < 3; ++d) if (fabs(R[6 + d]) < fabs(R[6 + k])) k = d;
    double a[3] = {0, 0, 0};
    a[k] = 1.0;
    const double dot = R[6 + k];
    double u[3], un = 0;
    for (int d = 0; d < 3; ++d) { u[d] = a[d] - dot * R[6 + d]; un += u[d] * u[d]; }
    un = sqrt(un);
    for (int d = 0; d < 3; ++d) R[d] = u[d] / un;
    R[3] = R[7] * R[2] - R[8] * R[1]; R[4] = R[8] * R[0] - R[6] * R[2]; R[5] = R[6] * R[1] - R[7] * R[0];   // e_v = e_w x e_u
  }
  for (int64_t i = 0; i < n_pix; ++i) {
    const double x = pix[i], y = pix[(size_t)n_pix + i], z = pix[(size_t)2 * n_pix + i];
    for (int d = 0; d < 3; ++d) pix[(size_t)d * n_pix + i] = R[3 * d] * x + R[3 * d + 1] * y + R[3 * d + 2] * z;
  }
}

// Grids of one (input cell, output cell) pair from the cells' bounding boxes (x in wavelengths, r as pixel coordinates).
void pair_geometry(const double* xlo, const double* xhi, const double* rlo, const double* rhi, int w, CellGeom& g, int64_t& n1, int64_t& n2) {
  n1 = 1; n2 = 1;
  for (int d = 0; d < 3; ++d) {
    const double xl = xlo[d], xu = xhi[d];
    const double sl = -6.283185307179586 * rhi[d], su = -6.283185307179586 * rlo[d];
    g.xc[d] = 0.5 * (xl + xu); g.sc[d] = 0.5 * (sl + su);
    const double X = std::max(0.5 * (xu - xl), 1e-9), S = std::max(0.5 * (su - sl), 1e-9);
    // at least one grid point per unit of X S beyond the minimum, so that degenerate (thin) dimensions stay tiny
    const double XS = std::max(X * S, 0.5);
    const double S_eff = XS / X;                                    // S widened when X S is tiny: theta stays within +-pi/sigma
    g.nf1[d] = next_smooth_even(std::max(2 * w, (int)ceil(2.0 * kSigma * X * S_eff / 3.141592653589793) + w + 2));
    g.nf2[d] = next_smooth_even(std::max(2 * w, (int)ceil(kSigma * g.nf1[d])));
    g.pos_scale[d] = kSigma * S_eff / 3.141592653589793;
    g.theta_scale[d] = 3.141592653589793 / (kSigma * S_eff);
    n1 *= g.nf1[d]; n2 *= g.nf2[d];
  }
}

int kernel_width(double eps) { return std::min(kMaxW, std::max(2, (int)ceil(-log10(eps / 10.0)) + 1)); }

}  // namespace

extern "C" int bb_nufft_destroy(bb_nufft* h) {
  if (!h) return BB_OK;
  cudaSetDevice(bb_ctx_device(h->ctx));
  cudaStreamSynchronize(bb_ctx_user_stream(h->ctx));
  for (auto& kv : h->plans) cufftDestroy(kv.second.handle);
  for (auto& kv : h->dec) cudaFree(kv.second);
  cudaFree(h->fft_work); cudaFree(h->lam_full); cudaFree(h->B_full); cudaFree(h->D_full);
  cudaFree(h->pix_dev); cudaFree(h->img); cudaFree(h->out_idx_dev); cudaFree(h->V); cudaFree(h->grid); cudaFree(h->fine);
  cudaFree(h->in_idx_dev); cudaFree(h->xyz_all_dev); cudaFree(h->inv_wl_dev); cudaFree(h->B_dev); cudaFree(h->D_dev); cudaFree(h->xyz_dev);
  bb_ctx_ref(h->ctx, -1);
  delete h;
  return BB_OK;
}

extern "C" int bb_nufft_create(bb_ctx* ctx, int64_t n_pix, const double* pix, int64_t ld_pix, int n_levels, double eps,
                               int n_part_in, int n_part_out, bb_nufft** out) {
  if (!out) return BB_EINVAL;
  *out = nullptr;
  if (!ctx || n_pix < 1 || n_pix > 0x7fffffff || !pix || ld_pix < n_pix || n_levels < 1 || n_levels > BB_MAX_LEVELS ||
      !(eps >= 1e-7 && eps <= 1e-2) || n_part_in < 1 || n_part_in > 64 || n_part_out < 1 || n_part_out > 64)
    return BB_EINVAL;
  BB_CUDA(cudaSetDevice(bb_ctx_device(ctx)));
  bb_nufft* h = new (std::nothrow) bb_nufft;
  if (!h) return BB_EALLOC;
  h->ctx = ctx; h->n_pix = n_pix; h->pix_stride = (n_pix + 63) / 64 * 64; h->n_levels = n_levels;
  bb_ctx_ref(ctx, +1);
  h->n_part_in = n_part_in; h->n_part_out = n_part_out;
  // kernel width from the tolerance (one more grid point per decade, as FINUFFT's rule for sigma = 2), beta = 2.30 w
  h->kp.w = kernel_width(eps);
  h->kp.beta = 2.30 * h->kp.w;
  double gx[kQuad], gw[kQuad];
  gauss_legendre_01(gx, gw);
  cudaStream_t st = bb_ctx_user_stream(ctx);
  int rc = BB_OK;
  do {
    if (cudaMemcpyToSymbol(c_gl_x, gx, sizeof(gx)) != cudaSuccess || cudaMemcpyToSymbol(c_gl_w, gw, sizeof(gw)) != cudaSuccess) { rc = BB_ECUDA; break; }
    h->pix_host.resize((size_t)3 * n_pix);
    if (cudaStreamSynchronize(st) != cudaSuccess ||
        cudaMemcpy2D(h->pix_host.data(), n_pix * sizeof(double), pix, ld_pix * sizeof(double), n_pix * sizeof(double), 3,
                     cudaMemcpyDefault) != cudaSuccess) { rc = BB_ECUDA; break; }
    if (cudaMalloc(&h->pix_dev, (size_t)3 * n_pix * sizeof(double)) != cudaSuccess ||
        cudaMalloc(&h->img, (size_t)n_levels * h->pix_stride * sizeof(float)) != cudaSuccess ||
        cudaMalloc(&h->out_idx_dev, (size_t)n_pix * sizeof(int)) != cudaSuccess) { rc = BB_EALLOC; break; }
    rotate_to_mean_direction(h->pix_host, n_pix, h->R);
    std::vector<int> order;
    partition(h->pix_host.data(), n_pix, n_pix, n_part_out, h->out_start, order, h->out_lo, h->out_hi);
    if (cudaMemcpy(h->pix_dev, h->pix_host.data(), (size_t)3 * n_pix * sizeof(double), cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMemcpy(h->out_idx_dev, order.data(), (size_t)n_pix * sizeof(int), cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMemset(h->img, 0, (size_t)n_levels * h->pix_stride * sizeof(float)) != cudaSuccess) { rc = BB_ECUDA; break; }
  } while (0);
  if (rc != BB_OK) { cudaGetLastError(); bb_nufft_destroy(h); return rc; }
  *out = h;
  return BB_OK;
}

constexpr int64_t kMaxPendingSources = (int64_t)1 << 24;   // host bookkeeping: 24 B of coordinates + 4 B of index per staged baseline

constexpr size_t kMaxCachedPlans = 64, kMaxCachedDec = 1024;

// One set of transforms over the baselines of all staged collects (Eq. 36 over cells; the sum over time steps is just more sources).
// Two passes. The first is host-only bookkeeping plus every allocation: the geometry of all (input cell, output cell)
// pairs, the grid limit, the grids and the shared FFT work area grown to the largest pair, the deconvolution arrays
// and the cuFFT plans. Whatever can refuse the flush (BB_EUNSUPPORTED, BB_EALLOC, plan creation) does so THERE, before
// a single kernel has added to the images: the staged collects are dropped, the images are as before the flush. The
// second pass only launches; an error in it is a CUDA launch or execution failure (BB_ECUDA), after which the images are
// undefined and the handle should be destroyed.
static int nufft_flush(bb_nufft* h) {
  if (h->pend == 0) return BB_OK;
  cudaStream_t st = bb_ctx_user_stream(h->ctx);
  const int L = h->n_levels, w = h->kp.w, n_ant = h->pend_n_ant, T = h->pend;
  const int64_t n_base = (int64_t)n_ant * n_ant, n_total = n_base * T;
  h->pend = 0;                                                          // whatever happens below, the staged collects are consumed
  int rc;
  if ((rc = grow(&h->in_idx_dev, &h->in_idx_cap, (size_t)n_total)) != BB_OK || (rc = grow(&h->xyz_all_dev, &h->xyz_all_cap, h->xyz_all.size())) != BB_OK ||
      (rc = grow(&h->inv_wl_dev, &h->inv_wl_cap, h->inv_wl_all.size())) != BB_OK)
    return rc;
  // baselines on the host for the cell bookkeeping (Section 3.4.1): coordinates only, no visibility values
  std::vector<double> bl((size_t)3 * n_total);
  for (int c = 0; c < T; ++c) {
    const double* xh = h->xyz_all.data() + (size_t)c * 3 * n_ant;
    const double iw = h->inv_wl_all[c];
    for (int d = 0; d < 3; ++d)
      for (int q = 0; q < n_ant; ++q)
        for (int p = 0; p < n_ant; ++p)
          bl[(size_t)d * n_total + (size_t)c * n_base + p + (size_t)n_ant * q] = (xh[(size_t)d * n_ant + p] - xh[(size_t)d * n_ant + q]) * iw;
  }
  std::vector<int> in_start, in_order;
  std::vector<double> in_lo, in_hi;
  partition(bl.data(), n_total, n_total, h->n_part_in, in_start, in_order, in_lo, in_hi);
  const int n_in = h->n_part_in * h->n_part_in, n_out = h->n_part_out * h->n_part_out;

  // ---- pass 1: geometry, limits, allocations, plans -------------------------------------------------
  struct Pair { int ic, oc; CellGeom g; int64_t n1, n2; const double* dec[3]; bb_nufft::FftPlan* plan; };
  std::vector<Pair> pairs;
  int64_t max_n1 = 0, max_n2 = 0;
  for (int ic = 0; ic < n_in; ++ic) {
    if (in_start[ic + 1] == in_start[ic]) continue;
    for (int oc = 0; oc < n_out; ++oc) {
      if (h->out_start[oc + 1] == h->out_start[oc]) continue;
      Pair pr{};
      pr.ic = ic; pr.oc = oc;
      pair_geometry(&in_lo[ic * 3], &in_hi[ic * 3], &h->out_lo[oc * 3], &h->out_hi[oc * 3], w, pr.g, pr.n1, pr.n2);
      if ((double)pr.n2 * L * 8.0 > kMaxGridBytes || pr.n2 > 0x7fffffffLL) return BB_EUNSUPPORTED;
      max_n1 = std::max(max_n1, pr.n1); max_n2 = std::max(max_n2, pr.n2);
      pairs.push_back(pr);
    }
  }
  double gx[kQuad], gw[kQuad];
  gauss_legendre_01(gx, gw);
  std::vector<double> dec;
  size_t work_need = 0;
  for (Pair& pr : pairs) {
    // 1 / phihat(2 pi m / nf2) per dimension (Eq. 35 for the inner type-2 step): one device array per (nf1, nf2), kept
    for (int d = 0; d < 3; ++d) {
      const auto dk = std::make_pair(pr.g.nf1[d], pr.g.nf2[d]);
      auto di = h->dec.find(dk);
      if (di == h->dec.end()) {
        dec.resize((size_t)pr.g.nf1[d]);
        for (int i = 0; i < pr.g.nf1[d]; ++i) dec[i] = 1.0 / es_hat_host(6.283185307179586 * (i - pr.g.nf1[d] / 2) / pr.g.nf2[d], h->kp, gx, gw);
        double* dp = nullptr;
        if (cudaMalloc(&dp, dec.size() * sizeof(double)) != cudaSuccess) { cudaGetLastError(); return BB_EALLOC; }
        di = h->dec.emplace(dk, dp).first;                             // owned by the handle from here on
        BB_CUDA(cudaMemcpy(dp, dec.data(), dec.size() * sizeof(double), cudaMemcpyHostToDevice));
      }
      pr.dec[d] = di->second;
    }
    const auto key = std::make_tuple(pr.g.nf2[0], pr.g.nf2[1], pr.g.nf2[2]);
    auto it = h->plans.find(key);
    if (it == h->plans.end()) {
      bb_nufft::FftPlan fp{};
      int dims[3] = {pr.g.nf2[2], pr.g.nf2[1], pr.g.nf2[0]};           // slowest first
      if (cufftCreate(&fp.handle) != CUFFT_SUCCESS) return BB_ECUDA;
      if (cufftSetAutoAllocation(fp.handle, 0) != CUFFT_SUCCESS ||
          cufftMakePlanMany(fp.handle, 3, dims, nullptr, 1, 0, nullptr, 1, 0, CUFFT_C2C, 1, &fp.work_bytes) != CUFFT_SUCCESS) {
        cufftDestroy(fp.handle);
        return BB_ECUDA;
      }
      it = h->plans.emplace(key, fp).first;
    }
    pr.plan = &it->second;                                              // std::map: stable under later insertions
    work_need = std::max(work_need, it->second.work_bytes);
  }
  // the FFT work area belongs to the same budget as the fine grids it serves
  if ((double)max_n2 * L * 8.0 + (double)work_need > kMaxGridBytes) return BB_EUNSUPPORTED;
  if ((rc = grow(&h->grid, &h->grid_cap, (size_t)L * max_n1)) != BB_OK || (rc = grow(&h->fine, &h->fine_cap, (size_t)L * max_n2)) != BB_OK ||
      (rc = grow(&h->fft_work, &h->fft_work_cap, std::max(work_need, (size_t)256))) != BB_OK)
    return rc;                                                          // (cudaFree of a buffer in use waits for the device)

  // ---- pass 2: launches only -----------------------------------------------------------------------
  auto run = [&]() -> int {
    BB_CUDA(cudaMemcpyAsync(h->xyz_all_dev, h->xyz_all.data(), h->xyz_all.size() * sizeof(double), cudaMemcpyHostToDevice, st));
    BB_CUDA(cudaMemcpyAsync(h->inv_wl_dev, h->inv_wl_all.data(), h->inv_wl_all.size() * sizeof(double), cudaMemcpyHostToDevice, st));
    BB_CUDA(cudaMemcpyAsync(h->in_idx_dev, in_order.data(), (size_t)n_total * sizeof(int), cudaMemcpyHostToDevice, st));
    for (const Pair& pr : pairs) {
      const int n_src = in_start[pr.ic + 1] - in_start[pr.ic], n_tgt = h->out_start[pr.oc + 1] - h->out_start[pr.oc];
      const int64_t n1 = pr.n1, n2 = pr.n2;
      BB_CUDA(cudaMemsetAsync(h->grid, 0, (size_t)L * n1 * sizeof(float2), st));
      BB_CUDA(cudaMemsetAsync(h->fine, 0, (size_t)L * n2 * sizeof(float2), st));
      spread_kernel<<<(unsigned)((n_src + 3) / 4), 128, 0, st>>>(h->in_idx_dev + in_start[pr.ic], n_src, h->xyz_all_dev, n_ant, h->inv_wl_dev,
                                                                    h->V, L, pr.g, h->kp, h->grid);
      BB_CUDA(cudaGetLastError());
      deconv_pad_kernel<<<(unsigned)((n1 + 255) / 256), 256, 0, st>>>(h->grid, L, pr.g, pr.dec[0], pr.dec[1], pr.dec[2], h->fine);
      BB_CUDA(cudaGetLastError());
      if (cufftSetStream(pr.plan->handle, st) != CUFFT_SUCCESS || cufftSetWorkArea(pr.plan->handle, h->fft_work) != CUFFT_SUCCESS) return BB_ECUDA;
      for (int l = 0; l < L; ++l)                                      // u_k = sum_m b_m exp(+i m k h2): the unnormalised inverse
        if (cufftExecC2C(pr.plan->handle, reinterpret_cast<cufftComplex*>(h->fine + (size_t)l * n2),
                         reinterpret_cast<cufftComplex*>(h->fine + (size_t)l * n2), CUFFT_INVERSE) != CUFFT_SUCCESS) return BB_ECUDA;
      interp_kernel<<<(unsigned)((n_tgt + 3) / 4), 128, 0, st>>>(h->out_idx_dev + h->out_start[pr.oc], n_tgt, h->pix_dev, h->n_pix,
                                                                    h->fine, L, pr.g, h->kp, h->img, h->pix_stride);
      BB_CUDA(cudaGetLastError());
      h->n_transforms += 1;
      h->max_grid = std::max(h->max_grid, n2);
    }
    return BB_OK;
  };
  rc = run();
  const cudaError_t e = cudaStreamSynchronize(st);                      // on every path: host vectors above are in flight until here
  if (rc == BB_OK && e != cudaSuccess) { bb_note_cuda_error(e, "bb_nufft flush", __FILE__, __LINE__); rc = BB_ECUDA; }
  if (h->plans.size() > kMaxCachedPlans) {
    for (auto& kv : h->plans) cufftDestroy(kv.second.handle);
    h->plans.clear();
  }
  if (h->dec.size() > kMaxCachedDec) {
    for (auto& kv : h->dec) cudaFree(kv.second);
    h->dec.clear();
  }
  return rc;
}

extern "C" int bb_nufft_collect_eig(bb_nufft* h, int n_ant, int n_eig, double wavelength, const bb_c32* B, int ldb,
                                    const float* D, int ldd, const double* xyz, int ldxyz) {
  if (!h || !B || !D || !xyz || n_ant < 1 || n_ant > 4096 || n_eig < 1 || n_eig > 4096 || !(wavelength > 0.0) || ldb < n_ant ||
      ldd < h->n_levels || ldxyz < n_ant)
    return BB_EINVAL;
  BB_CUDA(cudaSetDevice(bb_ctx_device(h->ctx)));
  cudaStream_t st = bb_ctx_user_stream(h->ctx);
  const int L = h->n_levels;
  const int64_t n_base = (int64_t)n_ant * n_ant;
  int rc;
  if (h->pend > 0 && (h->pend_n_ant != n_ant || (h->pend + 1) * n_base > kMaxPendingSources) && (rc = nufft_flush(h)) != BB_OK) return rc;
  if ((rc = grow(&h->B_dev, &h->B_cap, (size_t)n_ant * n_eig)) != BB_OK || (rc = grow(&h->D_dev, &h->D_cap, (size_t)L * n_eig)) != BB_OK ||
      (rc = grow(&h->xyz_dev, &h->xyz_cap, (size_t)3 * n_ant)) != BB_OK)
    return rc;
  const size_t v_need = (size_t)(h->pend + 1) * L * n_base;
  if (v_need > h->V_cap) {                                            // grow and keep the staged collects' visibilities
    const size_t cap = std::max(v_need, 2 * h->V_cap);
    float2* nv = nullptr;
    if (cudaMalloc(&nv, cap * sizeof(float2)) != cudaSuccess) { cudaGetLastError(); return BB_EALLOC; }
    if (h->pend > 0) BB_CUDA(cudaMemcpyAsync(nv, h->V, (size_t)h->pend * L * n_base * sizeof(float2), cudaMemcpyDeviceToDevice, st));
    BB_CUDA(cudaStreamSynchronize(st));
    cudaFree(h->V);
    h->V = nv; h->V_cap = cap;
  }
  // snapshot the inputs (host or device: unified addressing), compact
  BB_CUDA(cudaMemcpy2DAsync(h->B_dev, (size_t)n_ant * 8, B, (size_t)ldb * 8, (size_t)n_ant * 8, n_eig, cudaMemcpyDefault, st));
  BB_CUDA(cudaMemcpy2DAsync(h->D_dev, (size_t)L * 4, D, (size_t)ldd * 4, (size_t)L * 4, n_eig, cudaMemcpyDefault, st));
  BB_CUDA(cudaMemcpy2DAsync(h->xyz_dev, (size_t)n_ant * 8, xyz, (size_t)ldxyz * 8, (size_t)n_ant * 8, 3, cudaMemcpyDefault, st));
  vis_kernel<<<(unsigned)((n_base + 255) / 256), 256, 0, st>>>(h->B_dev, n_ant, h->D_dev, L, n_ant, n_eig, L,
                                                               h->V + (size_t)h->pend * L * n_base);
  BB_CUDA(cudaGetLastError());
  std::vector<double> xh((size_t)3 * n_ant);
  BB_CUDA(cudaMemcpyAsync(xh.data(), h->xyz_dev, xh.size() * sizeof(double), cudaMemcpyDeviceToHost, st));
  BB_CUDA(cudaStreamSynchronize(st));
  if (h->pend == 0) { h->xyz_all.clear(); h->inv_wl_all.clear(); }
  const size_t o = h->xyz_all.size();
  h->xyz_all.resize(o + (size_t)3 * n_ant);
  for (int p = 0; p < n_ant; ++p) {                                   // antenna positions into the handle's rotated frame
    const double x = xh[p], y = xh[(size_t)n_ant + p], z = xh[(size_t)2 * n_ant + p];
    for (int d = 0; d < 3; ++d) h->xyz_all[o + (size_t)d * n_ant + p] = h->R[3 * d] * x + h->R[3 * d + 1] * y + h->R[3 * d + 2] * z;
  }
  h->inv_wl_all.push_back(1.0 / wavelength);
  h->pend += 1; h->pend_n_ant = n_ant;
  return BB_OK;
}

// Algorithm 3 as the paper states it: from S, W, the antenna positions and the intervals. Lines 2-4
// (Gram matrix, generalized eigendecomposition, N_eig largest) are the library's fp64 device glue (bb_eig), lines 6-7 the
// level weights (bb_level_weights: interval selection and filter in one matrix D), line 8 onwards bb_nufft_collect_eig
// (V = alpha_I diag(lambda_f) alpha_I^H per level with the beamforming folded in, B = W alpha, Eq. 17 / 21; then the NUFFT).
// The intermediates stay on the device.
extern "C" int bb_nufft_collect(bb_nufft* h, int n_ant, int n_beam, int n_eig, double wavelength, const bb_c32* W, int ldw,
                                const bb_c32* S, int lds, const double* xyz, int ldxyz, const double* intervals, int ld_int,
                                int n_filters, const int* filters) {
  if (!h || !S || !xyz || !intervals || !filters || n_filters < 1 || n_filters > BB_MAX_FILTERS || h->n_levels % n_filters != 0)
    return BB_EINVAL;
  const int n_intervals = h->n_levels / n_filters;
  if (n_ant < 1 || n_ant > 4096 || n_beam < 1 || n_beam > BB_MAX_BEAMS || n_eig < 1 || n_eig > n_beam || !(wavelength > 0.0) || lds < n_beam ||
      ldxyz < n_ant || ld_int < n_intervals || (W && ldw < n_ant) || (!W && n_beam != n_ant))
    return BB_EINVAL;
  BB_CUDA(cudaSetDevice(bb_ctx_device(h->ctx)));
  int rc;
  if ((rc = grow(&h->lam_full, &h->lam_full_cap, (size_t)n_eig)) != BB_OK || (rc = grow(&h->B_full, &h->B_full_cap, (size_t)n_ant * n_eig)) != BB_OK ||
      (rc = grow(&h->D_full, &h->D_full_cap, (size_t)h->n_levels * n_eig)) != BB_OK)
    return rc;
  // l.2-4 (+ B = W alpha). Synchronous; BB_ENOTPOSDEF / BB_ENOCONV come back directly and nothing is staged.
  if ((rc = bb_eig(h->ctx, n_ant, n_beam, n_eig, wavelength, W, ldw, S, lds, xyz, ldxyz, h->lam_full, h->B_full, n_ant)) != BB_OK) return rc;
  // l.5-7: D[f * n_intervals + i, k] = filter_f(lambda_k) if lambda_k lies in interval i, else 0
  if ((rc = bb_level_weights(h->ctx, h->lam_full, n_eig, intervals, ld_int, n_intervals, n_filters, filters, h->D_full, h->n_levels)) != BB_OK)
    return rc;
  // l.8-9: per-level visibilities and the (staged) type-3 transform
  return bb_nufft_collect_eig(h, n_ant, n_eig, wavelength, h->B_full, n_ant, h->D_full, h->n_levels, xyz, ldxyz);
}

extern "C" int bb_nufft_get(bb_nufft* h, int level, float* out) {
  if (!h || !out || level < 0 || level >= h->n_levels) return BB_EINVAL;
  BB_CUDA(cudaSetDevice(bb_ctx_device(h->ctx)));
  cudaStream_t st = bb_ctx_user_stream(h->ctx);
  int rc = nufft_flush(h);
  if (rc != BB_OK) return rc;
  BB_CUDA(cudaMemcpyAsync(out, h->img + (size_t)level * h->pix_stride, (size_t)h->n_pix * sizeof(float), cudaMemcpyDefault, st));
  BB_CUDA(cudaStreamSynchronize(st));
  return BB_OK;
}

extern "C" int bb_nufft_stats(bb_nufft* h, int64_t* n_transforms, int64_t* max_grid_points) {
  if (!h) return BB_EINVAL;
  if (n_transforms) *n_transforms = h->n_transforms;
  if (max_grid_points) *max_grid_points = h->max_grid;
  return BB_OK;
}


// Host-only: what Section 3.4.1 / Figure 1c-d is about — the transforms one collect would need, without running them.
extern "C" int bb_nufft_plan(int64_t n_pix, const double* pix, int64_t ld_pix, int n_ant, const double* xyz, int ldxyz, double wavelength,
                             double eps, int n_part_in, int n_part_out, int64_t* n_transforms, int64_t* max_grid_points,
                             double* sum_grid_points, double* nonempty_input_cells) {
  if (n_pix < 1 || n_pix > 0x7fffffff || !pix || ld_pix < n_pix || n_ant < 1 || n_ant > 4096 || !xyz || ldxyz < n_ant || !(wavelength > 0.0) ||
      !(eps >= 1e-7 && eps <= 1e-2) || n_part_in < 1 || n_part_in > 64 || n_part_out < 1 || n_part_out > 64)
    return BB_EINVAL;
  std::vector<double> ph((size_t)3 * n_pix);
  for (int d = 0; d < 3; ++d) for (int64_t i = 0; i < n_pix; ++i) ph[(size_t)d * n_pix + i] = pix[(size_t)d * ld_pix + i];
  double R[9] = {1, 0, 0, 0, 1, 0, 0, 0, 1};
  rotate_to_mean_direction(ph, n_pix, R);
  std::vector<int> out_start, order, in_start, in_order;
  std::vector<double> out_lo, out_hi, in_lo, in_hi;
  partition(ph.data(), n_pix, n_pix, n_part_out, out_start, order, out_lo, out_hi);
  const int64_t n_base = (int64_t)n_ant * n_ant;
  std::vector<double> xr((size_t)3 * n_ant), bl((size_t)3 * n_base);
  for (int p = 0; p < n_ant; ++p)
    for (int d = 0; d < 3; ++d) xr[(size_t)d * n_ant + p] = R[3 * d] * xyz[p] + R[3 * d + 1] * xyz[(size_t)ldxyz + p] + R[3 * d + 2] * xyz[(size_t)2 * ldxyz + p];
  for (int d = 0; d < 3; ++d)
    for (int q = 0; q < n_ant; ++q)
      for (int p = 0; p < n_ant; ++p) bl[(size_t)d * n_base + p + (size_t)n_ant * q] = (xr[(size_t)d * n_ant + p] - xr[(size_t)d * n_ant + q]) / wavelength;
  partition(bl.data(), n_base, n_base, n_part_in, in_start, in_order, in_lo, in_hi);
  const int w = kernel_width(eps), n_in = n_part_in * n_part_in, n_out = n_part_out * n_part_out;
  int64_t nt = 0, mx = 0, occupied = 0;
  double sum = 0.0;
  for (int ic = 0; ic < n_in; ++ic) {
    if (in_start[ic + 1] == in_start[ic]) continue;
    ++occupied;
    for (int oc = 0; oc < n_out; ++oc) {
      if (out_start[oc + 1] == out_start[oc]) continue;
      CellGeom g{};
      int64_t n1, n2;
      pair_geometry(&in_lo[ic * 3], &in_hi[ic * 3], &out_lo[oc * 3], &out_hi[oc * 3], w, g, n1, n2);
      ++nt; mx = std::max(mx, n2); sum += (double)n2;
    }
  }
  if (n_transforms) *n_transforms = nt;
  if (max_grid_points) *max_grid_points = mx;
  if (sum_grid_points) *sum_grid_points = sum;
  if (nonempty_input_cells) *nonempty_input_cells = (double)occupied / n_in;
  return BB_OK;
}
