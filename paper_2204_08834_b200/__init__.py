"""B200-native projection step of the FluTAS two-fluid method (arxiv 2204.08834, sec. 3.3)."""
