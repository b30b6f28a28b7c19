"""gk-b200: B200-native hot path of the local flux-tube delta-f gyrokinetic solver of
arxiv/paper_2604_06085 (field solve -> linear terms -> ExB bracket -> RK4 stage), as a C-ABI CUDA
library (libgk.so, include/gk.h) plus this thin ctypes binding.  PyTorch is used only for device
memory and streams.  There is no CPU fallback: importing works anywhere, every call needs CUDA."""
from .binding import (GkContext, GkError, lib_path, load_library, exported_symbols,  # noqa: F401
                      gk_spectra_static, gk_spectra_static_max,
                      T_I, T_II, T_IV, T_V, T_VII, T_VIII, T_DISS_S, T_DISS_V, T_HYP, T_III, T_ALL)

__all__ = ["GkContext", "GkError", "lib_path", "load_library", "exported_symbols",
           "gk_spectra_static", "gk_spectra_static_max"]
