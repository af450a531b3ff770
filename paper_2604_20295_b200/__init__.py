"""B200-native ETac tactile hot path (arxiv/paper_2604_20295): C-ABI library + thin binding."""
