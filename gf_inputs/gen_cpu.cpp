// Host build of the synthetic gauge-field generator (see gen_core.h for the recipe).  Input tooling only.
#include "gen_core.h"

#include <cstdint>

using namespace gfin;

template <class T>
static void gen_sites(T* out, const int* n, double r, uint64_t seed, const int64_t* sites, int64_t nsites) {
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < nsites; ++i) {
    int64_t site = sites ? sites[i] : i;
    m3 g0 = gauge_at(seed, (uint64_t)site);
    for (int mu = 0; mu < 4; ++mu) {
      m3 g1 = gauge_at(seed, (uint64_t)neighbour_up(site, mu, n));
      m3 e = smooth_link(seed, (uint64_t)site, mu, r);
      store_link(out + (i * 4 + mu) * 18, finish_link(g0, e, g1));
    }
  }
}

extern "C" {

// Whole field (sites == NULL, nsites == V) or the 4 links of each listed site, canonical layout, prec: 0 = f64, 1 = f32.
int gfin_links_host(void* out, const int* dims, double roughness, uint64_t seed, const int64_t* sites,
                    int64_t nsites, int prec) {
  if (!out || !dims) return -1;
  if (prec == 0) gen_sites((double*)out, dims, roughness, seed, sites, nsites);
  else if (prec == 1) gen_sites((float*)out, dims, roughness, seed, sites, nsites);
  else return -1;
  return 0;
}

// The hidden gauge rotation G(x) for the listed sites (or all): out[site][3][3][2], always f64.
int gfin_gauge_host(double* out, const int* dims, uint64_t seed, const int64_t* sites, int64_t nsites) {
  if (!out || !dims) return -1;
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < nsites; ++i) {
    int64_t site = sites ? sites[i] : i;
    store_link(out + i * 18, gauge_at(seed, (uint64_t)site));
  }
  return 0;
}

}  // extern "C"
