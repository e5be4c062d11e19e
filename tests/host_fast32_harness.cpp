// Host build of the fp32 production arithmetic (csrc/gl_fast32.cuh compiles as plain C++ with exact
// libm in place of the MUFU approximations): lets the CPU test suite check steps a3 + a4 of the
// CUDA path against the oracle without a GPU.  Test infrastructure only.
#include <cmath>
#include "../paper_2410_05408_b200/csrc/gl_fast32.cuh"
#include "../paper_2410_05408_b200/csrc/gl_tables.h"

extern "C" int host_flux_geometry_f32(const double* geom, long long n, double* flux_out) {
    float p32[8], o32[8];
    glt::smoothed_gauss_legendre<float>(16, p32, o32);
    static glf::TrapNode trap[16];
    for (int k = 0; k < 8; ++k) {
        glf::c_gl_phi[k] = p32[k];
        glf::c_gl_om[k] = o32[k];
    }
    for (int k = 0; k < 16; ++k) {
        trap[k].c = glf::c_trap_cos[k] = (float)cosl(3.141592653589793238462643383279502884L * k / 16);
        trap[k].s = glf::c_trap_sin[k] = (float)sinl(3.141592653589793238462643383279502884L * k / 16);
    }
    trap[8].c = 0.f;
    trap[0].s = 0.f;
    for (long long i = 0; i < n; ++i) {
        const double d = geom[6 * i], Rp = geom[6 * i + 1], fp = geom[6 * i + 2], pa = geom[6 * i + 3];
        const double u1 = geom[6 * i + 4], u2 = geom[6 * i + 5];
        const double pn = 3.14159265358979323846 * (1.0 - u1 / 3.0 - u2 / 6.0);
        float s, c;
        sincosf((float)pa, &s, &c);
        const float delta = glf::blocked_f32(trap, (float)d * c, -(float)d * s, (float)Rp,
                                             (float)(Rp * (1.0 - fp)), (float)((1.0 - u1 - 2.0 * u2) / pn),
                                             (float)((u1 + 2.0 * u2) / pn), (float)(u2 / pn));
        flux_out[i] = 1.0 - (double)delta;
    }
    return 0;
}

// The tables of the library's generator (gl_tables.h), for the check of the literal copies that
// csrc/gl_hot.cuh carries as immediates: phi8, om8 = smoothed 16-point Gauss-Legendre; trap32 =
// (cos, sin)(pi k / 16), k = 0..15, interleaved.
extern "C" void host_tables(float* phi8, float* om8, float* trap32) {
    glt::smoothed_gauss_legendre<float>(16, phi8, om8);
    for (int k = 0; k < 16; ++k) {
        trap32[2 * k] = (float)cosl(3.141592653589793238462643383279502884L * k / 16);
        trap32[2 * k + 1] = (float)sinl(3.141592653589793238462643383279502884L * k / 16);
    }
    trap32[16] = 0.f;   // exact zeros at the axes, as the library sets them
    trap32[1] = 0.f;
}
