"""paper_2606_16359_b200 -- B200-native (sm_100a) hot path of FEnc^2 (arxiv/paper_2606_16359): a CKKS homomorphic
convolution layer over fragment-encoded ciphertexts, as hand-written CUDA kernels behind the C ABI of include/fenc.h.

`binding` is argument marshalling only.  There is no CPU fallback and nothing here imports oracle/."""
from .binding import (Ciphertext, Context, ConvDesc, FcDesc, FcInfo, FencError, Keys, Layout, ParamsDesc, Plaintext, RELIN_KEY_ID,  # noqa: F401
                      SYMBOLS, Weights, load_library)
