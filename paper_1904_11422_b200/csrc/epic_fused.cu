// placeholder: fused path not built yet
#include "epic_internal.h"
namespace epic {
int fused_plan_init(epic_plan* p) { p->fused_ok = 0; p->d_fused = nullptr; return EPIC_OK; }
void fused_plan_free(epic_plan* p) { (void)p; }
int fused_supported(const epic_plan* p, int is_cf32, int n_pol, int n_products) { (void)p; (void)is_cf32; (void)n_pol; (void)n_products; return 0; }
int fused_image(epic_plan* p, const ImageArgs& a) { (void)p; (void)a; return EPIC_ERR_RANGE; }
}
