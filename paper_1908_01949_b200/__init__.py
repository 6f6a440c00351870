"""B200-native brute-force track-seed scan for a cylindrical drift chamber
(hot path of arXiv 1908.01949).  See DESIGN.md."""
