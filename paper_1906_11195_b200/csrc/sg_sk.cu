// sg_sk.cu -- Sherrington-Kirkpatrick path (row a4 of SURVEY.md 8(a); PAPER.md:43 Eq. 1, :233).
#include "sg_sim.h"

int sg_sk_create_impl(sg_sim *) { sg_set_error("SK model: not built yet"); return SG_EINVAL; }
int sg_sk_sweep_impl(sg_sim *, uint64_t) { return SG_EINVAL; }
int sg_sk_energy_impl(sg_sim *, int64_t *) { return SG_EINVAL; }
int sg_sk_get_spins_impl(sg_sim *, const uint64_t *, uint64_t *) { return SG_EINVAL; }
int sg_sk_set_spins_impl(sg_sim *, const uint64_t *) { return SG_EINVAL; }
int sg_sk_get_couplings_impl(sg_sim *, uint64_t *) { return SG_EINVAL; }
