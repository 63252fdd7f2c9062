"""osc-b200: per-event three-flavour neutrino oscillation reweighting on one NVIDIA B200 (sm_100a, fp64).

The product is the C-ABI library ``libosc_b200.so`` (include/osc.h, sources under ``csrc/``); this
package is its thin Python binding (``binding.py``), its build step (``build.py``) and the seeded
synthetic input generators (``workloads.py``).  See DESIGN.md.
"""
from .binding import (  # noqa: F401
    N_CHANNELS, OscError, osc_bin_centre_compare, osc_bin_index, osc_fp64_issue_probe, osc_fp64_peak_probe, osc_get_device, osc_last_error, osc_launch_count, osc_neg2lnl, osc_plan_create, osc_plan_destroy, osc_plan_reweight_bin,
    osc_plan_reweight_bin_batch, OscPlan,
    osc_params, osc_prob, osc_prob_all, osc_prob_host, osc_reweight_bin, osc_reweight_bin_batch, osc_reweight_bin_scales,
    osc_reweight_bin_host, osc_reweight_bin_scales_host, osc_reweight_bin_static, osc_set_batch_path, osc_set_device, osc_set_k2_tuning, osc_set_params, osc_version, pack_params,
)
