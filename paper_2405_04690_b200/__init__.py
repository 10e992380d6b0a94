"""B200-native GB waveform + delta-lnL hot path of arxiv 2405.04690 ("Erebor").

The product is the C-ABI library libgbfit.so (include/gbfit.h, csrc/); this package is its thin
Python binding.  Names follow the header: Context.waveform / delta_loglike / residual_update.
"""
from .gbfit import (ADD, REMOVE, SWAP, Context, Data, GbError, EXPORTS, lib, lib_path, version)  # noqa: F401
from . import build  # noqa: F401  (module: build.build() compiles libgbfit.so)
