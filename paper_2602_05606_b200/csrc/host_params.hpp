// host_params.hpp -- host-side S0 (Table I lines 1-4) shared by the .cu launchers; see host_params.cpp.
#pragma once
#include "coefs.cuh"

namespace kappagen {
bool domain_ok(double kappa, double theta);                 // kappa > 3/2, theta >= 0, finite
TableIParams<double> host_table1(double kappa);             // rounded once from long double
Coef<float> host_coef_f32(double kappa, double theta, bool fold);   // fold: see coefs.cuh
Coef<double> host_coef_f64(double kappa, double theta);
void set_error(const char* fmt, ...);
}  // namespace kappagen
