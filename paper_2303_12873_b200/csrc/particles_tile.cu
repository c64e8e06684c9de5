// particles_tile.cu -- placeholder until the fused per-tile kernel lands: routes to the global path.
#include "pic_internal.h"
namespace pic {
int tile_setup() { return 0; }
int launch_particles_tile(const Grid& g, const Fields& f, const Particles& p, long long n, double q, double m,
                          int order, const unsigned int*, DevStatus* status, cudaStream_t st) {
    launch_particles_global(g, f, p, n, q, m, order, status, st);
    return 1;
}
}  // namespace pic
