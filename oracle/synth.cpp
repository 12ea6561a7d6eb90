// ORACLE — TEST INFRASTRUCTURE, NOT PRODUCT CODE.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
// legs may call this. It shares no code with paper_2310_09200_b200/csrc.
//
// oracle_synth: the Standard Synthesizer of Bluebild written out in fp64 exactly in the
// loop order of the paper's GEMMEXP kernel.
//
//   PAPER.md:313-343  Algorithm 2 "GEMMEXP": for pixel { for antenna { p <- exp(i 2pi/lambda
//                     <P_icrs[a], X_pix[p]>); for eig: R[e] += p * U[a,e] } for eig:
//                     E[e,p] += |R[e]|^2 }
//   PAPER.md:121-125  Eq. 15  eps_aj = sum_p exp(-2 pi i f/c <x_p, r_j>) alpha_ap
//   PAPER.md:154-157  Eq. 20  I_{i0,in} = sum_{a in level} lambda_a |eps_a|^2
//   PAPER.md:294-306  Algorithm 1 lines 6-12: B^(ni,nf) += sum_{i in K} d_f^(i) E^(i)
//
// Readings: U = W*alpha = B (Q2); R is zeroed for every
// pixel (Q2); lambda in Alg. 2 is the wavelength (Q2, Q3); the contraction is
// E_kj = sum_i conj(B_ik) exp(+j 2 pi <p_i, r_j>/lambda_w) (Q1: the data model of Eq. 3
// has exp(+...), and Eq. 15 is its complex conjugate - same modulus); the level/filter
// weights arrive as the dense matrix D[l,k] (= lambda_k if lambda_k lies in interval l,
// else 0, for the LSQ filter) so that Alg. 1 line 9 is I_l += sum_k D[l,k] |E_k|^2.
//
// Layout (all column-major, as PAPER.md:270 states for the inputs of Table 1):
//   B    complex128, n_ant x n_eig, leading dimension ldb (interleaved re,im)
//   D    float64,    n_levels x n_eig, leading dimension ldd
//   xyz  float64,    n_ant x 3, leading dimension ldxyz   (metres)
//   pix  float64,    n_pix x 3, leading dimension ldpix   (unit vectors, same frame)
//   img  float64,    n_levels images of n_pix, img[l*n_pix + j], accumulated into (+=)
//
// Threads split the pixel range; pixels are independent so this changes no arithmetic.
#include <complex>
#include <cmath>
#include <thread>
#include <vector>
#include <cstdint>

namespace {

void synth_range(int n_ant, int n_eig, int n_levels, int64_t n_pix, int64_t j0, int64_t j1,
                 const std::complex<double>* B, int ldb, const double* D, int ldd,
                 const double* xyz, int ldxyz, const double* pix, int64_t ldpix,
                 double wavelength, double* img) {
    const double two_pi_over_lambda = 2.0 * M_PI / wavelength;
    std::vector<std::complex<double>> R(n_eig);
    for (int64_t j = j0; j < j1; ++j) {                        // Alg. 2 line 2
        for (int k = 0; k < n_eig; ++k) R[k] = 0.0;            // (Q2) reset per pixel
        const double rx = pix[j], ry = pix[j + ldpix], rz = pix[j + 2 * ldpix];
        for (int i = 0; i < n_ant; ++i) {                      // Alg. 2 line 4
            const double dot = xyz[i] * rx + xyz[i + ldxyz] * ry + xyz[i + 2 * ldxyz] * rz;
            const double phi = two_pi_over_lambda * dot;       // Alg. 2 line 5
            const std::complex<double> p(std::cos(phi), std::sin(phi));
            for (int k = 0; k < n_eig; ++k)                    // Alg. 2 lines 6-7
                R[k] += std::conj(B[i + (int64_t)k * ldb]) * p;
        }
        for (int k = 0; k < n_eig; ++k) {                      // Alg. 2 lines 10-12
            const double e = std::norm(R[k]);                  // |R|^2
            for (int l = 0; l < n_levels; ++l)                 // Alg. 1 line 9 / Eq. 20
                img[(int64_t)l * n_pix + j] += D[l + (int64_t)k * ldd] * e;
        }
    }
}

}  // namespace

extern "C" int oracle_synth(int n_ant, int n_eig, int n_levels, int64_t n_pix,
                            const double* B, int ldb, const double* D, int ldd,
                            const double* xyz, int ldxyz, const double* pix, int64_t ldpix,
                            double wavelength, double* img, int n_threads) {
    if (n_ant < 0 || n_eig < 0 || n_levels < 0 || n_pix < 0 || !(wavelength > 0.0)) return 1;
    if (n_threads <= 0) n_threads = (int)std::thread::hardware_concurrency();
    if (n_threads <= 0) n_threads = 1;
    if ((int64_t)n_threads > n_pix) n_threads = n_pix > 0 ? (int)n_pix : 1;
    const auto* Bc = reinterpret_cast<const std::complex<double>*>(B);
    std::vector<std::thread> pool;
    for (int t = 0; t < n_threads; ++t) {
        const int64_t j0 = n_pix * t / n_threads, j1 = n_pix * (t + 1) / n_threads;
        pool.emplace_back(synth_range, n_ant, n_eig, n_levels, n_pix, j0, j1, Bc, ldb, D, ldd,
                          xyz, ldxyz, pix, ldpix, wavelength, img);
    }
    for (auto& th : pool) th.join();
    return 0;
}

extern "C" int oracle_hardware_threads() { return (int)std::thread::hardware_concurrency(); }
