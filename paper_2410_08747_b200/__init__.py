"""B200-native hot path of McXtrace-style X-ray ray tracing (arxiv 2410.08747): a C-ABI CUDA library
(include/mcx.h, csrc/) and its thin ctypes binding.  See DESIGN.md."""
from .binding import Instrument, McxError, lib, probe_dfma, probe_l2, probe_latency, probe_tally  # noqa: F401
from .build import build  # noqa: F401
