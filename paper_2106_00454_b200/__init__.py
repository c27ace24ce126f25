"""B200-native (sm_100a) WPCD hot path: thin ctypes binding over the C-ABI library in csrc/ (see include/wpcd.h).

`from paper_2106_00454_b200 import wpcd` loads libwpcd.so and fails loudly if it is missing.  There is no CPU
fallback.  `paper_2106_00454_b200.inputs` (seeded synthetic inputs) has no dependency on the library.
"""
