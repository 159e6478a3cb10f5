"""B200-native superphoton transport (GPUmonty-style relativistic Monte Carlo radiative transfer)."""
