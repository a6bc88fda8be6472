"""B200-native hot path of the BITS method (arXiv 1208.3407): place -> sort -> search -> reduce."""
