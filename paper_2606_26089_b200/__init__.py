"""pd: B200-native (sm_100a) Delphes-style detector-response hot path behind a C ABI (include/pd.h).

`binding` marshals torch tensors into libpd.so; every step of the chain runs in its CUDA kernels.
There is no CPU fallback."""
from . import binding  # noqa: F401
from .binding import (Card, DeviceEFlow, DeviceImpact, DeviceTrackRefs, DeviceEvents, DeviceFeatures, DeviceMerged, DeviceObjects, DeviceOutputs, HostBuffers, PdError, last_launch_count, last_status,  # noqa: F401
                      event_features, filter_eflow, pileup_merge, pileup_status, card_upload, simulate, simulate_host, track_impact, truth_features, truth_features_static, workspace_bytes)
