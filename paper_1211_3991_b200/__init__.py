"""B200-native hot path of arXiv 1211.3991: coloured Metropolis + over-relaxation + parallel tempering
for the XY model on dilute Levy graphs.  See DESIGN.md."""
