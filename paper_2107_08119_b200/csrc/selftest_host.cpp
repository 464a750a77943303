// selftest_host.cpp -- CPU check of nep_math.cuh (build box, no GPU): the harmonic basis against
// Legendre polynomials (addition theorem), ylm_force and radial_fn against central differences.
// Built and run by tests/test_host_math.py:  g++ -O1 -o selftest_host selftest_host.cpp && ./selftest_host
#include <cstdio>
#include <cstdlib>
#include <cmath>
#include "nep_math.cuh"
using namespace nepk;

static double legendre(int l, double c) {
    double p0 = 1, p1 = c;
    if (l == 0) return 1;
    for (int k = 1; k < l; ++k) { double p2 = ((2 * k + 1) * c * p1 - k * p0) / (k + 1); p0 = p1; p1 = p2; }
    return p1;
}
static double urand() { return rand() / (double)RAND_MAX; }
static void unit(double* v) {
    double n;
    do { for (int a = 0; a < 3; ++a) v[a] = 2 * urand() - 1; n = sqrt(v[0]*v[0]+v[1]*v[1]+v[2]*v[2]); } while (n < 0.1 || n > 1);
    for (int a = 0; a < 3; ++a) v[a] /= n;
}

int main() {
    srand(7);
    int fails = 0;
    const int lof[kNumLM] = {NEP_LOF_LIST};
    // 1. addition theorem
    for (int t = 0; t < 200; ++t) {
        double u[3], v[3]; unit(u); unit(v);
        float bu[kNumLM], bv[kNumLM];
        ylm_basis((float)u[0], (float)u[1], (float)u[2], bu);
        ylm_basis((float)v[0], (float)v[1], (float)v[2], bv);
        double c = u[0]*v[0]+u[1]*v[1]+u[2]*v[2];
        for (int l = 1; l <= 4; ++l) {
            double s = 0; for (int m = 0; m < kNumLM; ++m) if (lof[m] == l) s += clm(m) * bu[m] * bv[m];
            if (fabs(s - legendre(l, c)) > 2e-5) { printf("addition theorem l=%d %g vs %g\n", l, s, legendre(l, c)); ++fails; }
        }
    }
    // 2. radial_fn against the definition in double + central differences
    for (int t = 0; t < 200; ++t) {
        const double rc = 4.0 + urand() * 2, r = 0.3 + urand() * (rc - 0.35), om = 1 + 60 * urand();
        float g[9], dg[9];
        radial_fn<9, true>((float)r, (float)(1 / rc), (float)om, g, dg);
        auto G = [&](double rr, int n) { double x = 2*(rr/rc-1)*(rr/rc-1)-1; return 0.5*(cos(n*acos(x))+1)*0.5*(1+cos(M_PI*rr/rc))*om; };
        for (int n = 0; n < 9; ++n) {
            double ref = G(r, n), h = 1e-5, dref = (G(r + h, n) - G(r - h, n)) / (2 * h);
            if (fabs(g[n] - ref) > 3e-6 * om) { printf("g[%d] r=%g %g vs %g\n", n, r, g[n], ref); ++fails; }
            if (fabs(dg[n] - dref) > 3e-5 * om) { printf("dg[%d] r=%g %g vs %g\n", n, r, dg[n], dref); ++fails; }
        }
    }
    // 3. ylm_force == gradient of Phi(rvec) = sum_m a_m(r) b_m(rvec/r), a_m(r) = alpha_m + beta_m r
    for (int t = 0; t < 100; ++t) {
        double alpha[kNumLM], beta[kNumLM], u[3]; unit(u);
        const double r = 1.5 + 2 * urand();
        for (int m = 0; m < kNumLM; ++m) { alpha[m] = 2*urand()-1; beta[m] = 2*urand()-1; }
        auto Phi = [&](const double* R) {
            double rr = sqrt(R[0]*R[0]+R[1]*R[1]+R[2]*R[2]); float b[kNumLM];
            // basis in double through a double re-evaluation of the same polynomials
            double x = R[0]/rr, y = R[1]/rr, z = R[2]/rr;
            double c2=x*x-y*y,s2=2*x*y,c3=x*c2-y*s2,s3=x*s2+y*c2,z2=z*z;
            double B[kNumLM]={x,y,z,3*z2-1,x*z,y*z,c2,s2,z*(5*z2-3),x*(5*z2-1),y*(5*z2-1),z*c2,z*s2,c3,s3,
                35*z2*z2-30*z2+3,x*z*(7*z2-3),y*z*(7*z2-3),c2*(7*z2-1),s2*(7*z2-1),z*c3,z*s3,c2*c2-s2*s2,2*c2*s2};
            (void)b; double s = 0; for (int m = 0; m < kNumLM; ++m) s += (alpha[m] + beta[m]*rr) * B[m]; return s; };
        float Sp[kNumLM], St[kNumLM];
        for (int m = 0; m < kNumLM; ++m) { St[m] = (float)((alpha[m] + beta[m]*r) / r); Sp[m] = (float)(beta[m] - lof[m] * (alpha[m] + beta[m]*r) / r); }
        float px, py, pz;
        ylm_force((float)u[0], (float)u[1], (float)u[2], Sp, St, &px, &py, &pz);
        double P[3] = {px, py, pz};
        for (int a = 0; a < 3; ++a) {
            double Rp[3] = {u[0]*r, u[1]*r, u[2]*r}, Rm[3] = {u[0]*r, u[1]*r, u[2]*r}; const double h = 1e-5;
            Rp[a] += h; Rm[a] -= h;
            double ref = (Phi(Rp) - Phi(Rm)) / (2 * h);
            if (fabs(P[a] - ref) > 2e-4) { printf("ylm_force comp %d: %g vs %g\n", a, P[a], ref); ++fails; }
        }
    }
    // 4. tanh / sech^2
    for (double a = -12; a <= 12; a += 0.37) {
        float t, d; tanh_sech2((float)a, &t, &d);
        if (fabs(t - tanh(a)) > 2e-7 || fabs(d - 1 / (cosh((double)(float)a) * cosh((double)(float)a))) > 2e-6 * (1 / (cosh(a)*cosh(a))) + 1e-30) { printf("tanh %g\n", a); ++fails; }
    }
    // 5. half-split forms == the full forms (basis slices, gradient halves, radial_g / radial_gd)
    for (int t = 0; t < 200; ++t) {
        double u[3]; unit(u);
        const float x = (float)u[0], y = (float)u[1], z = (float)u[2];
        float b[kNumLM], h0[kHalfLM], h1[kHalfLM], St[kNumLM], Sq[kNumLM], zero[kNumLM] = {0};
        ylm_basis(x, y, z, b);
        ylm_basis_half<0>(x, y, z, h0);
        ylm_basis_half<1>(x, y, z, h1);
        for (int k = 0; k < kHalfLM; ++k) {
            if (fabs(h0[k] - b[half_m<0>(k)]) > 2e-6) { printf("basis half0 %d\n", k); ++fails; }
            if (fabs(h1[k] - b[half_m<1>(k)]) > 2e-6) { printf("basis half1 %d\n", k); ++fails; }
            if (half_l<0>(k) != lof[half_m<0>(k)] || half_l<1>(k) != lof[half_m<1>(k)]) { printf("half_l %d\n", k); ++fails; }
        }
        for (int m = 0; m < kNumLM; ++m) { St[m] = (float)(2 * urand() - 1); Sq[m] = 0.f; }
        float px, py, pz, ax, ay, az, bx, by, bz, S0[kHalfLM], S1[kHalfLM];
        ylm_force(x, y, z, zero, St, &px, &py, &pz);          // Sq = 0: only V
        for (int k = 0; k < kHalfLM; ++k) { S0[k] = St[half_m<0>(k)]; S1[k] = St[half_m<1>(k)]; }
        ylm_grad_half<0>(x, y, z, S0, &ax, &ay, &az);
        ylm_grad_half<1>(x, y, z, S1, &bx, &by, &bz);
        if (fabs(ax + bx - px) > 2e-5 || fabs(ay + by - py) > 2e-5 || fabs(az + bz - pz) > 2e-5) {
            printf("grad halves: %g %g %g vs %g %g %g\n", ax + bx, ay + by, az + bz, px, py, pz); ++fails; }
        const double rc = 4.0 + urand() * 2, r = 0.3 + urand() * (rc - 0.35), om = 1 + 60 * urand();
        float g[9], dg[9], g2[9], gs[9], dg2[9];
        radial_fn<9, true>((float)r, (float)(1 / rc), (float)om, g, dg);
        radial_g<9>((float)r, (float)(1 / rc), (float)om, g2);
        radial_gd<9>((float)r, (float)(1 / rc), (float)om, (float)(1 / r), gs, dg2);
        for (int n = 0; n < 9; ++n) {
            if (fabs(g2[n] - g[n]) > 2e-6 * om) { printf("radial_g[%d] %g vs %g\n", n, g2[n], g[n]); ++fails; }
            if (fabs(gs[n] * r - g[n]) > 2e-6 * om) { printf("radial_gd gs[%d] %g vs %g\n", n, gs[n] * r, g[n]); ++fails; }
            if (fabs(dg2[n] - dg[n]) > 2e-5 * om) { printf("radial_gd dg[%d] %g vs %g\n", n, dg2[n], dg[n]); ++fails; }
        }
    }
    printf(fails ? "FAILED %d\n" : "OK\n", fails);
    return fails ? 1 : 0;
}
