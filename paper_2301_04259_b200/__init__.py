"""B200-native disk-integrated stellar spectrum synthesis (the hot path of SOAP-GPU, arXiv:2301.04259).

The product is the C-ABI library ``libsoap_b200.so`` (include/soap_b200.h, sources in ``csrc/``);
this package is its thin Python binding.  ``from paper_2301_04259_b200 import binding`` raises if the
library has not been built - there is no CPU fallback and the CPU oracle is never imported from here.
"""
from . import binding  # noqa: F401
from .binding import (  # noqa: F401
    Spectra, Star, SoapError,
    soap_create, soap_destroy, soap_set_option, soap_get_stats,
    soap_disk_geometry, soap_integrate_quiet, soap_integrate_quiet_static, soap_active_timeseries, soap_active_timeseries_effects,
    soap_export_geometry, soap_lower_resolution, soap_active_timeseries_evolving, soap_line_rvs,
    soap_synthesize_host, soap_batch_disk_geometry, soap_batch_integrate_quiet, soap_batch_active_timeseries, soap_contrast_planck,
    to_device_spectra,
)
