// Host build of the CUDA library's double-double Newell primitives (csrc/dd.cuh, newell_dd.cuh)
// so that tests/test_dd_host.py can check them on a box without a GPU.  Test-only.
#define HFFT_DD_HOST_TEST 1
#include "../paper_1910_07054_b200/csrc/newell_dd.cuh"

extern "C" {
void hfft_test_phi6(const double x[2], const double y[2], const double z[2], double out[12]) {
    hfft::dd phi[6];
    hfft::newell_phi6(hfft::dd_make(x[0], x[1]), hfft::dd_make(y[0], y[1]), hfft::dd_make(z[0], z[1]), phi);
    for (int c = 0; c < 6; ++c) { out[2 * c] = phi[c].hi; out[2 * c + 1] = phi[c].lo; }
}
void hfft_test_log(const double a[2], double out[2]) {
    hfft::dd r = hfft::dd_log(hfft::dd_make(a[0], a[1]));
    out[0] = r.hi; out[1] = r.lo;
}
void hfft_test_atan(const double a[2], double out[2]) {
    hfft::dd r = hfft::dd_atan_pos(hfft::dd_make(a[0], a[1]));
    out[0] = r.hi; out[1] = r.lo;
}
void hfft_test_sqrt_div(const double a[2], const double b[2], double out[4]) {
    hfft::dd r = hfft::dd_sqrt(hfft::dd_make(a[0], a[1]));
    hfft::dd q = hfft::dd_div(hfft::dd_make(a[0], a[1]), hfft::dd_make(b[0], b[1]));
    out[0] = r.hi; out[1] = r.lo; out[2] = q.hi; out[3] = q.lo;
}
}
