// ltjk_laplace.cpp -- step a3 (placeholder until the Remez solver lands; returns LTJK_ENOCONV, never a fake grid)
#include "../../include/ltjk.h"
extern "C" int ltjk_laplace_quadrature(double, double, int, double*, double*, double*) { return LTJK_ENOCONV; }
