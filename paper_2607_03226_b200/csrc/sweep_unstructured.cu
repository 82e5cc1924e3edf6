// sweep_unstructured.cu -- placeholder until the level-scheduled unstructured path lands.
#include "host_util.h"

int nb_launch_sweep_unstructured(nanobte_solver *h) { return nb_fail(h, NANOBTE_E_UNSUPPORTED, "unstructured sweep not built yet"); }
int nb_launch_moments_unstructured(nanobte_solver *h) { return nb_fail(h, NANOBTE_E_UNSUPPORTED, "unstructured moments not built yet"); }
int nb_launch_update_unstructured(nanobte_solver *h, int) { return nb_fail(h, NANOBTE_E_UNSUPPORTED, "unstructured update not built yet"); }
void nb_free_unstructured(nanobte_solver *) {}

extern "C" int nanobte_workspace_bytes_unstructured(const nanobte_unstructured_mesh *, const nanobte_bands *,
                                                    const nanobte_quadrature *, const nanobte_tag *, int32_t,
                                                    const nanobte_options *, size_t *) {
  return NANOBTE_E_UNSUPPORTED;
}
extern "C" int nanobte_create_unstructured(const nanobte_unstructured_mesh *, const nanobte_bands *, const nanobte_quadrature *,
                                           const nanobte_tag *, int32_t, const double *, const nanobte_options *, nanobte_solver **out) {
  if (!out) return NANOBTE_E_INVALID;
  nanobte_solver *h = new (std::nothrow) nanobte_solver();
  *out = h;
  return nb_fail(h, NANOBTE_E_UNSUPPORTED, "unstructured meshes not built yet");
}
