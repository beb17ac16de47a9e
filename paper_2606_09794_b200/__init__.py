"""B200-native NASGabor / SH-3 per-Gaussian colour evaluation (arxiv/paper_2606_09794).

``paper_2606_09794_b200.workloads``  seeded synthetic inputs (numpy only, no method arithmetic)
``paper_2606_09794_b200.build``      nvcc build of the C-ABI library (sm_100a)
``paper_2606_09794_b200.binding``    thin ctypes binding of ``include/nasg.h`` (loads the .so, fails
                                     loudly when it is missing; there is no CPU fallback)
"""
__version__ = "0.1.0"
