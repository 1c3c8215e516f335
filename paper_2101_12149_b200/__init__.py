"""B200-native electromagnetic PIC step (sort + gather + Boris push + Esirkepov deposit + Yee)
behind the C ABI of include/pic.h. The Python layer only marshals arguments; PyTorch is used by
callers for device memory and streams. No CPU fallback exists: use of any call without a built
libpic.so or without a CUDA device raises."""
from .binding import *  # noqa: F401,F403
from .binding import Sim, PicError, lib, LIB_PATH, SYMBOLS  # noqa: F401
