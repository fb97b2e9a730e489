"""B200-native event-based Monte Carlo neutron transport hot path (arxiv 2501.05440).

``inputs``  -- seeded synthetic problem generators (shared with the test oracle; no method arithmetic)
``binding`` -- thin ctypes binding of the C-ABI CUDA library (include/mcdc.h); loaded lazily so that
               importing the generators never needs the built extension.
"""


def __getattr__(name):
    if name in ("Problem", "load_library", "build", "McdcError"):
        from . import binding
        return getattr(binding, name)
    raise AttributeError(name)
