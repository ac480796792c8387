"""B200-native implicit, adaptive, charge-conserving PIC particle mover (arXiv 1111.5295):
CUDA kernels + C-ABI in csrc/ (include/pic.h), ctypes binding in binding.py, seeded workloads
in workloads.py.  Importing the package does not load the CUDA library; binding.load() does."""
