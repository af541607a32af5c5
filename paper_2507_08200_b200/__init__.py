"""paper_2507_08200_b200 -- B200-native (sm_100a) variable-coefficient geometric multigrid, the elliptic-solve
hot path of Vidyut3d (arxiv 2507.08200).  C-ABI library: include/vmg.h; binding: .binding."""
