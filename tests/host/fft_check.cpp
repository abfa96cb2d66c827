// Host build of the register FFT building blocks of csrc/pty_fft128.cuh (fft32 in both directions, the FMA-form
// radix-4 stage and its table) compared with a float64 DFT written out as a double loop.  The packed FP32x2
// intrinsics are replaced by their plain definitions; everything else is the device source, unchanged.
// Built and run by tests/test_host_fft.py (CPU, g++).
#define PTY_PORT_INCLUDED
#include <vector_types.h>
#include <vector_functions.h>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <complex>
#define PTY_DEV inline
inline float2 __fadd2_rn(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
inline float2 __fmul2_rn(float2 a, float2 b) { return make_float2(a.x * b.x, a.y * b.y); }
inline float2 __ffma2_rn(float2 a, float2 b, float2 c) { return make_float2(fmaf(a.x, b.x, c.x), fmaf(a.y, b.y, c.y)); }
namespace pty {
inline void pty_cta_sync() {}
inline void pty_cluster_sync() {}
inline void tmem_fence_before_sync() {}
inline void tmem_fence_after_sync() {}
inline void tmem_wait_st() {}
inline void tmem_wait_ld() {}
inline void tmem_st8(unsigned, const float2 (&)[32], int) {}
inline void tmem_ld8(unsigned, float2 (&)[32], int) {}
inline void sincospi(double x, double* s, double* c) { *s = sin(M_PI * x); *c = cos(M_PI * x); if (fabs(*c) < 1e-15) *c = 0; if (fabs(*s) < 1e-15) *s = 0; }
inline void sincospi_f(float x, float* s, float* c) { *s = (float)sin(M_PI * (double)x); *c = (float)cos(M_PI * (double)x); }
}
#include "pty_fft128.cuh"
using namespace pty;
typedef std::complex<double> cd;
template <int DIR> double check32() {
    float2 v[32]; cd x[32];
    for (int i = 0; i < 32; ++i) { v[i] = make_float2(drand48() - 0.5, drand48() - 0.5); x[i] = cd(v[i].x, v[i].y); }
    NoBg bg; fft32<DIR, 0>(v, bg);
    double err = 0, nrm = 0;
    for (int k = 0; k < 32; ++k) {
        cd s = 0; for (int n = 0; n < 32; ++n) s += x[n] * std::polar(1.0, DIR * 2 * M_PI * n * k / 32.0);
        err += std::norm(s - cd(v[k].x, v[k].y)); nrm += std::norm(s);
    }
    return sqrt(err / nrm);
}
void check_r4() {
    double worst = 0;
    for (int gi = 0; gi < 32; ++gi) {
        float e[12]; fill_twf(gi, e);
        float4 A = make_float4(e[0], e[1], e[2], e[3]), B = make_float4(e[4], e[5], e[6], e[7]), C = make_float4(e[8], e[9], e[10], e[11]);
        for (int rep = 0; rep < 20; ++rep) {
            float2 a[4]; cd x[4];
            for (int q = 0; q < 4; ++q) { a[q] = make_float2(drand48() - 0.5, drand48() - 0.5);
                x[q] = cd(a[q].x, a[q].y) * std::polar(1.0, -2 * M_PI * q * gi / 128.0); }
            bfly4_tw_fma(A, B, C, a[0], a[1], a[2], a[3]);
            double err = 0, nrm = 0;
            for (int k = 0; k < 4; ++k) {
                cd s = 0; for (int q = 0; q < 4; ++q) s += x[q] * std::polar(1.0, -2 * M_PI * q * k / 4.0);
                err += std::norm(s - cd(a[k].x, a[k].y)); nrm += std::norm(s);
            }
            worst = fmax(worst, sqrt(err / nrm));
        }
    }
    printf("radix-4 FMA form, worst rel err over gi: %.3e\n", worst);
}

int main() {
    srand48(1);
    printf("fft32 fwd rel err %.3e\n", check32<-1>());
    printf("fft32 inv rel err %.3e\n", check32<+1>());
    check_r4();
    return 0;
}
