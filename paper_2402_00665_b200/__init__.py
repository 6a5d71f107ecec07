"""B200-native linear BVH (modified Apetrei build + stackless range queries), arXiv 2402.00665.

``binding`` holds the thin ctypes layer over the C-ABI library ``libbvh_b200.so`` (include/bvh_b200.h);
``workloads`` the seeded input generators.  Nothing here imports ``oracle``.
"""
__all__ = ["binding", "workloads"]
