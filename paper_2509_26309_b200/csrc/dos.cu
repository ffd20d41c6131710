// dos.cu -- NEXT-1 of SURVEY 8(f): density of states from the correlation function (Analyzer.calc_dos).
// The paper gives no formula; the reading (#27) is a Hann-windowed direct Fourier transform of the state-averaged
// correlation with C_0 = 1 and C_{-n} = conj(C_n).  Tiny next to the propagation: (2 n_step + 1) x n_step x n_state terms.
#include <cmath>

#include "tbpm_internal.h"

using namespace tbpm_detail;

namespace {

__global__ void k_dos(const double2 *__restrict__ corr, int n_state, int n_step, double dt, double rescale, double *energy,
                      double *dos)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j > 2 * n_step) return;
    const double E = -rescale + (double)j * (rescale / (double)n_step);
    const double inv_b = 1.0 / (double)n_state;
    double sum = 0.0;
    for (int n = 1; n <= n_step; ++n) {
        double cr = 0.0, ci = 0.0;                          // state average of C_n (entry n-1: t = n dt)
        for (int b = 0; b < n_state; ++b) {
            const double2 c = corr[(size_t)b * n_step + (n - 1)];
            cr += c.x;
            ci += c.y;
        }
        const double w = 0.5 * (1.0 + cospi((double)n / (double)n_step));
        double sn, cs;
        sincos((double)n * E * dt, &sn, &cs);
        sum += w * inv_b * (cr * cs - ci * sn);             // Re[C_n exp(+i n E dt)]
    }
    energy[j] = E;
    dos[j] = dt / (2.0 * 3.14159265358979323846) * (1.0 + 2.0 * sum);
}

}  // namespace

extern "C" int tbpm_dos(const double *corr, int n_state, int n_step, double dt, double rescale, double *energy, double *dos,
                        void *stream)
{
    if (n_state < 0 || n_step < 0 || !(rescale > 0.0) || !(dt > 0.0)) return TBPM_EINVAL;
    if (n_state == 0 || n_step == 0) return TBPM_OK;
    if (!corr || !energy || !dos) return TBPM_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const int n_e = 2 * n_step + 1, threads = 128;
    k_dos<<<(n_e + threads - 1) / threads, threads, 0, st>>>(reinterpret_cast<const double2 *>(corr), n_state, n_step, dt, rescale,
                                                             energy, dos);
    count_launches(1);
    TBPM_CUDA_TRY(cudaGetLastError());
    return TBPM_OK;
}

// NEXT-2, last step: LDOS from the Haydock coefficients by the continued fraction (reading #29)
//     G(z) = 1 / (z - a_0 - b_1^2 / (z - a_1 - b_2^2 / ( ... - b_{n-1}^2 / (z - a_{n-1})))),  z = E + i eta,  ldos = -Im G / pi,
// evaluated from the bottom up; one thread per (site, energy).  a, b as written by tbpm_haydock (b[.][n] = b_{n+1}).
namespace {
__global__ void k_haydock_ldos(const double *__restrict__ a, const double *__restrict__ b, int n_site, int n_iter, const double *__restrict__ energy,
                               int n_e, double eta, double *ldos)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n_site * n_e) return;
    const int s = t / n_e, j = t - s * n_e;
    const double zr = energy[j], zi = eta;
    double gr = 0.0, gi = 0.0;                               // G of the levels below
    for (int n = n_iter - 1; n >= 0; --n) {
        const double bb = n < n_iter - 1 ? b[(size_t)s * n_iter + n] : 0.0;
        const double dr = zr - a[(size_t)s * n_iter + n] - bb * bb * gr, di = zi - bb * bb * gi;
        const double m = dr * dr + di * di;
        gr = dr / m;
        gi = -di / m;
    }
    ldos[t] = -gi / 3.14159265358979323846;
}
}  // namespace

extern "C" int tbpm_haydock_ldos(const double *a, const double *b, int n_site, int n_iter, const double *energy, int n_energy, double eta,
                                 double *ldos, void *stream)
{
    if (n_site < 0 || n_iter < 1 || n_energy < 0 || !(eta > 0.0)) return TBPM_EINVAL;
    if (n_site == 0 || n_energy == 0) return TBPM_OK;
    if (!a || !b || !energy || !ldos) return TBPM_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const int total = n_site * n_energy, threads = 128;
    k_haydock_ldos<<<(total + threads - 1) / threads, threads, 0, st>>>(a, b, n_site, n_iter, energy, n_energy, eta, ldos);
    count_launches(1);
    TBPM_CUDA_TRY(cudaGetLastError());
    return TBPM_OK;
}
