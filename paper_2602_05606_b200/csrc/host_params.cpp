// host_params.cpp -- step S0 on the host: Table I lines 1-4, once per call ("The first
// four lines are required only once").  Evaluated in long double (ln B through lgammal,
// PAPER.md:250) and rounded once, so the kernels' constants carry no error of their own.  Compiled by
// g++ (not nvcc) because of long double.  Also: the thread-local error text behind kappagen_last_error.
#include "host_params.hpp"

#include <cmath>
#include <cstdarg>
#include <cstdio>

#include "../../include/kappagen.h"

namespace kappagen {

static thread_local char g_error[512] = "";

void set_error(const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_error, sizeof(g_error), fmt, ap);
    va_end(ap);
}

bool domain_ok(double kappa, double theta) {
    return std::isfinite(kappa) && std::isfinite(theta) && kappa > 1.5 && theta >= 0.0;
}

static TableIParams<long double> table1_ld(double kappa) {
    const long double k = (long double)kappa, ks = k - 0.5L;
    const long double lnB = lgammal(1.5L) + lgammal(ks) - lgammal(ks + 1.5L);
    // Eq. (20) with the printed decimals as long double literals
    const long double c = (0.123L * k * k - 1.12L * k + 2.56L) / (k * k - 7.89L * k + 15.6L);
    return table1_params<long double>(k, lnB, c);
}

TableIParams<double> host_table1(double kappa) {
    const TableIParams<long double> P = table1_ld(kappa);
    TableIParams<double> D;
    D.kstar = (double)P.kstar; D.a = (double)P.a; D.b = (double)P.b; D.c = (double)P.c;
    return D;
}

Coef<float> host_coef_f32(double kappa, double theta, bool fold) {
    return make_coef_f32<long double>(table1_ld(kappa), (long double)theta, fold);
}

Coef<double> host_coef_f64(double kappa, double theta) {
    return make_coef_f64<long double>(table1_ld(kappa), (long double)theta);
}

}  // namespace kappagen

extern "C" int kappagen_params(double kappa, double* kappa_star, double* a, double* b, double* c) {
    if (!kappa_star || !a || !b || !c) {
        kappagen::set_error("kappagen_params: NULL output pointer");
        return KAPPAGEN_ENULL;
    }
    if (!kappagen::domain_ok(kappa, 0.0)) {
        kappagen::set_error("kappagen_params: kappa = %g is outside kappa > 3/2", kappa);
        return KAPPAGEN_EINVAL;
    }
    const kappagen::TableIParams<double> P = kappagen::host_table1(kappa);
    *kappa_star = P.kstar; *a = P.a; *b = P.b; *c = P.c;
    return KAPPAGEN_OK;
}

extern "C" const char* kappagen_last_error(void) { return kappagen::g_error; }
extern "C" int kappagen_version(void) { return 100; }
