// Host build of paper_1601_02063_b200/csrc/dmath.cuh for tests/test_dmath.py (the hardware seeds are
// replaced by truncated libm values; everything else is the code the kernels run).
#include "../paper_1601_02063_b200/csrc/dmath.cuh"
extern "C" {
void dm_eval(int op, int n, const double* x, double* y, double* y2) {
    for (int i = 0; i < n; ++i) {
        switch (op) {
            case 0: y[i] = ody::d_rcp(x[i]); break;
            case 1: y[i] = ody::d_rsqrt(x[i]); break;
            case 2: y[i] = ody::d_sqrt(x[i]); break;
            case 3: ody::d_sincos(x[i], y[i], y2[i]); break;
            case 4: y[i] = ody::d_exp(x[i]); break;
            case 5: y[i] = ody::d_expm1(x[i]); break;
            case 6: y[i] = ody::d_log(x[i]); break;
            case 10: y[i] = ody::f_exp(x[i]); break;
            case 11: y[i] = ody::f_expm1_nc(x[i]); break;
            case 12: y[i] = ody::f_log(x[i]); break;
        }
    }
}
}
