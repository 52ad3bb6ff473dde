"""B200-native (sm_100a) hot path of arxiv/paper_2606_01114: demagnetisation field by pruned
FFT convolution with the Newell tensor, exchange/anisotropy/Zeeman terms, LLG right-hand side
and RK4, behind the C ABI of include/mm_b200.h.  See DESIGN.md."""
from .binding import (DMI_BULK, DMI_INTERFACIAL, LIB_PATH, MM_F32, MM_F64, TERM_ANISOTROPY,  # noqa: F401
                      TERM_DEMAG, TERM_DMI, TERM_EXCHANGE, TERM_STT, TERM_ZEEMAN, Context, MMError,
                      load_library)
