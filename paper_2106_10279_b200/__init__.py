"""madflow-b200: B200-native LO Monte Carlo integrand hot path."""
