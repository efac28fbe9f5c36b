"""B200-native RT-TDDFT time step (arXiv 2410.09189): C-ABI CUDA library + thin Python binding.

``from paper_2410_09189_b200 import binding`` loads ``librt_tddft.so`` (built by ``build.py``) and fails
loudly if it is missing; there is no CPU fallback.  ``workloads`` (seeded synthetic inputs) imports nothing
from the CUDA path.
"""
