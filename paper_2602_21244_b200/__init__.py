"""B200-native neural DSMC collision step (arxiv 2602.21244): C-ABI CUDA library + thin binding.

``from paper_2602_21244_b200 import dsmc`` loads the sm_100a shared library (and fails
loudly when it is missing); ``workloads`` holds the seeded synthetic input generators.
"""
