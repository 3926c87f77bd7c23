"""B200-native combinatorial-summation (CoS) evaluation: ctypes binding `api` over the C-ABI library libcos_b200.so
(include/cos.h), its in-tree build script `build`, and the batch-sharding helpers `sharding`.  See DESIGN.md."""

__all__ = ["api", "build", "sharding"]
