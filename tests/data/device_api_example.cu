// A user kernel written against the public header only (include/rlxpp_device.cuh): Monte-Carlo
// estimate of pi with a data-dependent number of draws per thread (rejection of points outside a
// band), the situation of PAPER.md lines 172-176.  Compiled by tests/test_host_library.py to show
// that the header is self-contained; not part of the library.
#include "rlxpp_device.cuh"

__global__ void pi_kernel(rlxpp_view_t view, unsigned long long* hits, unsigned int tries) {
  const unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= view.n) return;
  rlxpp_dev::Stream g;
  g.load(view, i);
  unsigned long long h = 0;
  for (unsigned int t = 0; t < tries; t++) {
    const unsigned mask = __activemask();
    const double x = g.draw_coop(mask), y = g.draw_coop(mask);
    h += x * x + y * y < 1.0 ? 1u : 0u;
  }
  g.store(view, i);
  hits[i] = h;
}
