"""paper_1305_0708_b200 -- B200-native tree-level |M|^2 (hot path of arXiv:1305.0708)."""
