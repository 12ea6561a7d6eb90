// ORACLE — TEST INFRASTRUCTURE, NOT PRODUCT CODE (see synth.cpp header).
//
// oracle_brute: the literal definition, for tiny inputs only. Kept in its own translation
// unit with no helper shared with synth.cpp, a different loop nest (level, pixel, eigenpair,
// antenna) and the complex exponential evaluated inside the innermost loop through
// std::exp(complex) instead of cos/sin, so that it pins oracle_synth (pin P1).
//
//   I_l(r_j) = sum_k D[l,k] | sum_i conj(B_ik) exp(j 2 pi <p_i, r_j> / lambda_w) |^2
//   PAPER.md:121-125 (Eq. 15), PAPER.md:154-157 (Eq. 20), PAPER.md:110-115 (Eq. 13-14)
//
// Same layouts as oracle_synth; img is overwritten (=), not accumulated.
#include <complex>
#include <cstdint>

extern "C" int oracle_brute(int n_ant, int n_eig, int n_levels, int64_t n_pix,
                            const double* B, int ldb, const double* D, int ldd,
                            const double* xyz, int ldxyz, const double* pix, int64_t ldpix,
                            double wavelength, double* img) {
    typedef std::complex<double> cplx;
    const cplx* Bc = reinterpret_cast<const cplx*>(B);
    const double pi = 3.14159265358979323846264338327950288;
    for (int l = 0; l < n_levels; ++l)
        for (int64_t j = 0; j < n_pix; ++j) {
            double acc = 0.0;
            for (int k = 0; k < n_eig; ++k) {
                cplx e(0.0, 0.0);
                for (int i = 0; i < n_ant; ++i) {
                    double d = 0.0;
                    for (int c = 0; c < 3; ++c) d += xyz[i + (int64_t)c * ldxyz] * pix[j + c * ldpix];
                    e += std::conj(Bc[i + (int64_t)k * ldb]) * std::exp(cplx(0.0, 2.0 * pi * d / wavelength));
                }
                acc += D[l + (int64_t)k * ldd] * (e.real() * e.real() + e.imag() * e.imag());
            }
            img[(int64_t)l * n_pix + j] = acc;
        }
    return 0;
}
