#include <cstdio>
#include <cmath>
#include <cstdlib>
// Host build of the device logarithm of potentials.cuh (log_pos is __host__ __device__) against logl.
// Built and run by tests/test_abi_cpu.py::test_device_log_against_libm; prints the worst error in ulps.
#include "../paper_1201_5029_b200/csrc/potentials.cuh"
int main(){
  double worst=0; double wx=0; srand(1);
  for (long i=0;i<4000000;i++){
    double u = rand()/(double)RAND_MAX, v = rand()/(double)RAND_MAX;
    double x;
    int mode = i%4;
    if (mode==0) x = pow(10.0, -300 + 600*u);
    else if (mode==1) x = 0.5 + 1.5*u;           // near 1
    else if (mode==2) x = 1.0 + (u-0.5)*1e-6*v;  // very near 1
    else x = ldexp(0.70710678118654752440*(1+ (u-0.5)*1e-3), (int)(v*40)-20); // near the sqrt2 switch
    long double want = logl((long double)x);
    double got = pycool::log_pos(x);
    double ulp = fabs(nextafter((double)want, INFINITY) - (double)want);
    if (ulp==0) ulp = 4.9e-324;
    double err = fabsl((long double)got - want)/ulp;
    if (fabs((double)want) < 1e-300) continue;
    if (err>worst){worst=err;wx=x;}
  }
  printf("worst %.3f ulp at x=%.17g\n", worst, wx);
  double sub = 1e-310; printf("sub %.17g %.17g\n", pycool::log_pos(sub), log(sub));
  return 0;
}
