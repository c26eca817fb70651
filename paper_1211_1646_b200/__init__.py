"""B200-native checkerboard cell sweep (MPMC for hard disks, arxiv 1211.1646).

`inputs` is pure numpy and safe to import anywhere; `binding` loads the CUDA C-ABI library and fails
loudly when it is missing.
"""
