"""paper_1008_0135_b200 — B200-native ray-casting volume renderer (C-ABI library + thin binding).

`from paper_1008_0135_b200 import vr` loads the CUDA extension (libvr_b200.so) and fails loudly if
it is missing; `workloads` (seeded synthetic inputs) imports neither the extension nor oracle/.
"""
